"""The allocation-free entry point (include/mpr.h: mpr_energy_of_angles_noalloc) against the existing path.

mpr_energy_of_angles_noalloc computes the energy per bond e = H / N_GP (Eq. 2) of an angle field with
its partial sums in a file-scope `static __device__` array of the library instead of a caller's workspace.  The existing
path is a context's mpr_set_angles + mpr_energy (k_energy: fp32 bond terms from the unit vectors, fp64 sums in the
workspace).  Tolerance: 2e-6 absolute on e, the T2b tolerance of tests/test_gpu_parity.py.  Also held against the oracle.

This file is collected last (pytest --collect-only: test_zz_*), so that a failure here hides no other test under -x; it
passes alone in a fresh process and after the other tests (the scratch is shared by every call and keeps the last call's
contents: the calls below go large -> small -> large on purpose)."""
import numpy as np
import pytest

from paper_1811_01604_b200 import synth
from test_gpu_parity import _dev, _field, mpr, torch_cuda   # noqa: F401  (fixtures)

pytestmark = pytest.mark.gpu
TOL_E = 2e-6


def _existing_path(torch, mpr, z, m, q, seed, sweeps):
    """(angles [rows, cols] as a CUDA tensor, e per bond by mpr_energy) of a context's state after a few sweeps."""
    ctx = mpr.Mpr(_dev(torch, z), _dev(torch, m))
    ctx.set_params(0.05, seed=seed, q=q)
    if sweeps:
        ctx.sweep(sweeps, 2.0)
    phi = ctx.get_angles()[0].contiguous().clone()
    ctx.set_angles(phi[None])            # mpr_energy of exactly the exported angles
    e = ctx.energy()[0]
    ctx.close()
    return phi, e


def test_noalloc_energy_matches_the_existing_path_on_calls_in_a_row(torch_cuda, mpr, orc):
    torch = torch_cuda
    cases = []
    for rows, cols, q, sweeps, seed in ((700, 523, 0.5, 3, 1), (37, 53, 0.5, 0, 2), (700, 523, 0.5, 3, 1), (2, 2, 0.3, 0, 3),
                                        (1024, 1024, 0.5, 2, 4), (129, 1000, 0.125, 1, 5)):
        z, m = _field(rows, cols, 6.0, 0.5, 60 + seed)
        phi, e_ctx = _existing_path(torch, mpr, z, m, q, seed, sweeps)
        cases.append((phi, float(np.float32(q)), e_ctx))
    out = torch.empty(1, dtype=torch.float64, device="cuda")
    got = []
    for phi, q, e_ctx in cases:          # back to back on one stream: each call finds the previous call's scratch
        mpr.energy_of_angles_noalloc(phi, q, out=out)
        got.append(float(out.cpu()[0]))
    for (phi, q, e_ctx), e in zip(cases, got):
        assert e == pytest.approx(e_ctx, abs=TOL_E), (tuple(phi.shape), q)
        assert e == pytest.approx(orc.energy_per_bond(phi.cpu().numpy(), q), abs=1e-9), (tuple(phi.shape), q)
    assert got[0] == got[2]              # the same field twice, another call in between: bit for bit the same
    # two calls in a row without reading in between, then again: the result does not depend on what the scratch held
    a, b = torch.empty(1, dtype=torch.float64, device="cuda"), torch.empty(1, dtype=torch.float64, device="cuda")
    mpr.energy_of_angles_noalloc(cases[4][0], cases[4][1], out=a)
    mpr.energy_of_angles_noalloc(cases[1][0], cases[1][1], out=b)
    assert float(a.cpu()[0]) == got[4] and float(b.cpu()[0]) == got[1]


def test_noalloc_rejects_sizes_beyond_its_scratch(torch_cuda, mpr):
    torch = torch_cuda
    phi = torch.zeros((4, 8), dtype=torch.float32, device="cuda")
    out = torch.full((1,), 7.0, dtype=torch.float64, device="cuda")
    with pytest.raises(mpr.MprError) as e:          # checked on the host before anything is enqueued
        mpr.energy_of_angles_noalloc(phi, 0.5, out=out, rows=mpr.NOALLOC_MAX_ROWS + 1)
    assert e.value.name == "MPR_ERR_TOO_LARGE" and str(mpr.NOALLOC_MAX_ROWS) in str(e.value)
    for bad in (dict(rows=1), dict(cols=1), dict(cols=70000)):
        with pytest.raises(mpr.MprError) as e:
            mpr.energy_of_angles_noalloc(phi, 0.5, out=out, **bad)
        assert e.value.name == "MPR_ERR_ARG"
    with pytest.raises(mpr.MprError) as e:
        mpr.energy_of_angles_noalloc(phi, 0.7, out=out)
    assert e.value.name == "MPR_ERR_ARG"
    assert float(out.cpu()[0]) == 7.0               # outputs untouched on error
    # the largest size it takes: MPR_NOALLOC_MAX_ROWS rows (aligned spins: e = -1 exactly)
    tall = torch.full((mpr.NOALLOC_MAX_ROWS, 3), 1.25, dtype=torch.float32, device="cuda")
    assert float(mpr.energy_of_angles_noalloc(tall, 0.5).cpu()[0]) == -1.0
