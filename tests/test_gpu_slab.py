"""One grid cut into row blocks over several contexts (mpr_create_slab) against ONE
context on the whole grid, which tests/test_gpu_parity.py holds against the oracle.  The slabs run in threads of this
process on one GPU -- each thread makes the calls a rank would make, the transport between them is a barrier and
device-to-device copies -- so what is tested is the decomposition (global Philox site words, global Eq. 1 range, ghost
rows, own-row reductions, the library's loops with their callbacks), not a network.  Unmeasured on more than one GPU.

Because the random numbers are keyed by the site of the whole grid and every reduction that feeds a decision is exact
(integer counts) or agrees to rounding (the energy sum, used only for the slope's sign), the slabs' states must equal
the single context's BIT FOR BIT: after the equilibration (same stopping sweep, same a) and after the realizations."""
import threading

import numpy as np
import pytest

from paper_1811_01604_b200 import synth
from test_gpu_parity import _dev, _field, mpr, torch_cuda   # noqa: F401  (fixtures)

pytestmark = pytest.mark.gpu


class ThreadComm:
    """Transport between slabs that live in threads of one process."""

    def __init__(self, n):
        self.n, self.bar, self.slots = n, threading.Barrier(n, timeout=120), [None] * n

    def rank(self, r):
        comm = self

        class _Rank:
            def allreduce(self, values, op):
                comm.slots[r] = list(values)
                comm.bar.wait()
                cols = list(zip(*comm.slots))                       # every thread reduces in rank order: same bits
                out = [(sum, min, max)[op](c) for c in cols]
                comm.bar.wait()
                return out

            def exchange(self, send_up, recv_up, send_down, recv_down, stream):
                import torch
                stream.synchronize()
                comm.slots[r] = (send_up, send_down)
                comm.bar.wait()
                with torch.cuda.stream(stream):
                    if recv_up is not None:
                        recv_up.copy_(comm.slots[r - 1][1])
                    if recv_down is not None:
                        recv_down.copy_(comm.slots[r + 1][0])
                stream.synchronize()
                comm.bar.wait()

        return _Rank()


def _run_slabs(torch, mpr, z, m, bounds, T, params, steps):
    """bounds: row boundaries [0, b1, ..., rows]; steps(ctx) -> dict of numpy results.  One thread per slab."""
    rows = z.shape[0]
    n = len(bounds) - 1
    comm = ThreadComm(n)
    out, err = [None] * n, [None] * n

    def work(r):
        try:
            torch.cuda.set_device(0)
            stream = torch.cuda.Stream()
            with torch.cuda.stream(stream):
                first, cnt = mpr.slab_local_rows(rows, z.shape[1], bounds[r], bounds[r + 1])
                ctx = mpr.MprSlab(_dev(torch, z[first:first + cnt]), _dev(torch, m[first:first + cnt]), rows, bounds[r],
                                  bounds[r + 1], comm.rank(r), stream=stream)
                ctx.set_params(T, **params)
                res = steps(ctx)
                stream.synchronize()
                out[r] = {k: (v[0][ctx.own] if isinstance(v, np.ndarray) and v.ndim == 3 else v) for k, v in res.items()}
                if ctx.comm_error is not None:
                    raise ctx.comm_error
                ctx.close()
        except BaseException as e:          # noqa: BLE001
            err[r] = e
            if not isinstance(e, mpr.MprError):      # a status comes back on every slab alike: nobody is left waiting
                comm.bar.abort()

    threads = [threading.Thread(target=work, args=(r,)) for r in range(n)]
    for t in threads:
        t.start()
    for t in threads:
        t.join()
    for e in err:
        if e is not None and not isinstance(e, threading.BrokenBarrierError):
            raise e
    for e in err:
        if e is not None:
            raise e
    return out


def _steps(ctx):
    ctx.equilibrate()
    st = ctx.get_stats()[0]
    res = {"phi_eq": ctx.get_angles().cpu().numpy(), "sweeps": st.equil_sweeps, "a": st.a, "t": st.t, "e_last": st.e_last,
           "A_last": st.A_last, "energy": ctx.energy()[0]}
    ctx.simulate()
    res.update(pred=ctx.predict().cpu().numpy(), std=ctx.predict_std().cpu().numpy(), phi_end=ctx.get_angles().cpu().numpy(),
               t_end=ctx.get_stats()[0].t, n_free=ctx.get_stats()[0].n_free)
    return res


@pytest.mark.parametrize("rows,cols,bounds,s", [
    (200, 150, [0, 96, 200], 1),            # two slabs, multi-tile local grids
    (200, 150, [0, 60, 130, 200], 7),       # three slabs: the middle one has ghost rows on both sides; 7 = 4 + 3 sweeps per realization
    (96, 64, [0, 48, 96], 4),               # local grids that are a single tile each, the whole grid a single tile too
    (600, 260, [0, 300, 600], 5),           # 64-row tiles
])
def test_slabs_reproduce_the_single_context_bit_for_bit(torch_cuda, mpr, rows, cols, bounds, s):
    torch = torch_cuda
    z, m = _field(rows, cols, 7.0, 0.5, 1234 + rows)
    z = (50.0 + 10.0 * z).astype(np.float32)
    # the extremes of the data in different slabs, so that Eq. 1 needs the range over all of them
    m[2, 3] = 1; z[2, 3] = z.max() + 5.0
    m[rows - 3, 5] = 1; z[rows - 3, 5] = z.min() - 5.0
    T = synth.choose_T(z, m)
    params = dict(seed=99, equil_cap=120, M=5, sweeps_per_real=s)
    ref = mpr.Mpr(_dev(torch, z), _dev(torch, m))
    ref.set_params(T, **params)
    want = _steps(ref)
    ref.close()
    got = _run_slabs(torch, mpr, z, m, bounds, T, params, _steps)
    for r, g in enumerate(got):
        own = slice(bounds[r], bounds[r + 1])
        assert (g["sweeps"], g["a"], g["t"], g["t_end"], g["A_last"]) == (want["sweeps"], want["a"], want["t"], want["t_end"], want["A_last"])
        # the energy is a double sum of float row sums of the tiles: another tiling, another rounding (~1e-10); it feeds
        # only the sign of the fitted slope
        assert g["e_last"] == pytest.approx(want["e_last"], abs=2e-9) and g["energy"] == pytest.approx(want["energy"], abs=2e-9)
        for key in ("phi_eq", "phi_end", "pred", "std"):
            assert np.array_equal(g[key].view(np.uint32), want[key][0][own].view(np.uint32)), (r, key)
    assert sum(g["n_free"] for g in got) == want["n_free"]
    assert want["sweeps"] < 120          # the stopping rule ended the equilibration, not the cap


def test_slab_errors_are_judged_on_the_whole_grid(torch_cuda, mpr):
    """A slab without any sample is fine when another slab has some; a grid without prediction sites, with a non-finite
    sample or a constant sample set fails on EVERY slab alike; a failing callback is MPR_ERR_COMM."""
    torch = torch_cuda
    rows, cols, bounds = 64, 40, [0, 32, 64]
    z, m = _field(rows, cols, 5.0, 0.5, 77)

    def names(zz, mm):
        def steps(ctx):
            return {"ok": True}
        try:
            _run_slabs(torch, mpr, zz, mm, bounds, 0.05, dict(seed=1), steps)
            return "MPR_OK"
        except mpr.MprError as e:
            return e.name

    m2 = m.copy(); m2[:40] = 0                         # the upper slab (and its ghost rows) holds no sample
    assert names(z, m2) == "MPR_OK"
    assert names(z, np.ones_like(m)) == "MPR_ERR_NO_FREE"
    assert names(z, np.zeros_like(m)) == "MPR_ERR_NO_SAMPLES"
    z3 = z.copy(); z3[50, 7] = np.inf; m3 = m.copy(); m3[50, 7] = 1
    assert names(z3, m3) == "MPR_ERR_NONFINITE"
    assert names(np.full_like(z, 2.0), m) == "MPR_ERR_DEGENERATE_RANGE"

    class Broken:
        def allreduce(self, values, op):
            raise RuntimeError("link down")

        def exchange(self, *a):
            raise RuntimeError("link down")

    with pytest.raises(mpr.MprError) as e:
        mpr.MprSlab(_dev(torch, z[:40]), _dev(torch, m[:40]), rows, 0, 32, Broken())
    assert e.value.name == "MPR_ERR_COMM"
    with pytest.raises(mpr.MprError) as e:           # an odd first row would flip the checkerboard colours
        mpr.MprSlab(_dev(torch, z[23:64]), _dev(torch, m[23:64]), rows, 31, 64, Broken())
    assert e.value.name == "MPR_ERR_ARG"
