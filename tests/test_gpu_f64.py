"""Parity of the double-precision CUDA path (mpr64_* calls; Table 2) against the oracle
built with double storage (oracle/mpr_oracle64.py), through the C ABI.

Tolerances.  Both sides compute in double; the CUDA path updates unit vectors (cos q phi, sin q phi), the oracle
angles.  One update is ~30 double operations on numbers of order 1 (relative rounding 1.1e-16 each), the export
phi = atan2(v) / q doubles the error at q = 1/2: a few 1e-15 rad expected, 1e-11 rad asserted (T2).  A decision flip
needs |AP - r| below that, which does not happen at these sizes: no exceptions are allowed.  Energies per bond: 1e-13.
Bit-exact: z_min, z_max, Eq. 1 at the sample sites, the bitmask-dependent parts (sample sites returned untouched), and
the initial draw 2 pi u."""
import math

import numpy as np
import pytest

from paper_1811_01604_b200 import synth

pytestmark = pytest.mark.gpu

TWO_PI = 2.0 * math.pi
TOL_RAD = 1e-11


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("a CUDA device is required for -m gpu tests (no CPU fallback exists)")
    return torch


@pytest.fixture(scope="module")
def mpr(torch_cuda):
    from paper_1811_01604_b200 import mpr as binding
    binding.lib()
    return binding


@pytest.fixture(scope="module")
def orc64():
    from oracle import mpr_oracle64
    mpr_oracle64.lib()
    return mpr_oracle64


def _dev(torch, a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _field(rows, cols, ell, p_removed, seed):
    z = synth.grf(rows, cols, ell, "gaussian", seed).astype(np.float64)
    # make the data genuinely double: a float field would hide a float path somewhere
    z = z + 1e-9 * np.random.default_rng(seed + 5).standard_normal(z.shape)
    mask = synth.bernoulli_mask(rows, cols, p_removed, seed + 1)
    mask.flat[0] = 1; mask.flat[-1] = 0
    if mask.sum() < 2:
        mask.flat[1] = 1
    return z, mask


@pytest.mark.parametrize("rows,cols", [(64, 64), (37, 53), (2, 2), (2, 9), (129, 1000)])
def test_t1_transform_and_initial_state_bit_exact(torch_cuda, mpr, orc64, rows, cols):
    torch = torch_cuda
    z, m = _field(rows, cols, 6.0, 0.4, 100 + rows)
    ctx = mpr.Mpr64(_dev(torch, z), _dev(torch, m))
    ctx.set_params(0.05, seed=1234)
    phi_o, zmin, zmax = orc64.transform(z, m, 1234)
    assert ctx.get_transform() == (float(zmin), float(zmax))
    phi_g = ctx.get_angles().cpu().numpy()
    assert phi_g.dtype == np.float64 and np.array_equal(phi_g, phi_o)
    st = ctx.get_stats()
    assert st.n_free == int((m == 0).sum()) and st.n_samples == int(m.sum())
    assert ctx.energy() == pytest.approx(orc64.energy_per_bond(phi_o), abs=1e-13)
    ctx.close()


def _one_sweep(orc64, ctx, phi0, mask, q, T, a, seed, t, or_mode):
    torch = ctx._torch
    ctx.set_angles(torch.from_numpy(phi0).cuda())
    ctx.set_sweep_index(t)
    acc_g = ctx.sweep(1, a, count=True)
    got = ctx.get_angles().cpu().numpy()
    ref = phi0.copy()
    acc_o = orc64.sweep(ref, mask, q, T, a, seed, 0, t, or_mode)
    free = mask == 0
    assert np.array_equal(got[~free], ref[~free])
    assert np.abs(got - ref)[free].max() <= TOL_RAD
    assert acc_g == acc_o
    assert ctx.energy() == pytest.approx(orc64.energy_per_bond(ref, q), abs=1e-13)
    assert ctx.get_stats().t == t + 1


@pytest.mark.parametrize("name,L", [("cfg1", 64), ("cfg2", 256), ("cfg3", 256), ("cfg4", 512)])
def test_t2_one_sweep_from_equilibrated_oracle_state(torch_cuda, mpr, orc64, name, L):
    torch = torch_cuda
    w = synth.make_workload(name, L=L)
    z, m, T = w.truth[0].astype(np.float64), w.mask[0], float(w.T[0])
    p = orc64.Params(seed=w.seed, equil_cap=150)
    phi, _, _ = orc64.transform(z, m, p.seed)
    st = orc64.equilibrate(phi, m, T, p)
    ctx = mpr.Mpr64(_dev(torch, z), _dev(torch, m))
    ctx.set_params(T, seed=p.seed)
    for t in (st["t"], st["t"] + 1):                       # an even and an odd sweep index: both word pairs
        _one_sweep(orc64, ctx, phi, m, 0.5, T, st["a"], p.seed, t, 0)
        orc64.sweep(phi, m, 0.5, T, st["a"], p.seed, 0, t)
    ctx.close()


@pytest.mark.parametrize("rows,cols", [(2, 2), (2, 7), (7, 2), (3, 3), (37, 53), (64, 129), (2, 20001), (20000, 3)])
def test_t2_ragged_and_tiny_grids_hot_start(torch_cuda, mpr, orc64, rows, cols):
    torch = torch_cuda
    z, m = _field(rows, cols, 3.0, 0.5, 300 + rows * cols)
    ctx = mpr.Mpr64(_dev(torch, z), _dev(torch, m))
    ctx.set_params(0.3, seed=9)
    phi, _, _ = orc64.transform(z, m, 9)
    for t in range(3):
        _one_sweep(orc64, ctx, phi, m, 0.5, 0.3, 1.0, 9, t, 0)
        orc64.sweep(phi, m, 0.5, 0.3, 1.0, 9, 0, t)
    ctx.close()


@pytest.mark.parametrize("q,or_mode", [(0.5, 2), (0.5, 1), (0.3, 0), (0.3, 2), (0.125, 0)])
def test_t2_other_q_and_over_relaxation_modes(torch_cuda, mpr, orc64, q, or_mode):
    torch = torch_cuda
    z, m = _field(96, 80, 6.0, 0.5, 41)
    ctx = mpr.Mpr64(_dev(torch, z), _dev(torch, m))
    ctx.set_params(0.1, seed=21, q=q, or_mode=or_mode)
    q = float(np.float32(q))                               # mpr_params.q is a float: the value the library was given
    phi, _, _ = orc64.transform(z, m, 21)
    for t in range(4):
        orc64.sweep(phi, m, q, 0.1, 2.0, 21, 0, t, or_mode)
    _one_sweep(orc64, ctx, phi, m, q, 0.1, 2.0, 21, 4, or_mode)
    ctx.close()


def test_equilibration_controller_and_full_run_follow_the_oracle(torch_cuda, mpr, orc64):
    """Whole path on a cfg1-shaped grid: with no decision near its threshold the two double chains are the same chain,
    so the stopping sweep, a, the energy and the prediction agree (prediction: 1e-9 of the data range)."""
    torch = torch_cuda
    w = synth.make_workload("cfg1")
    z, m, T = w.truth[0].astype(np.float64), w.mask[0], float(w.T[0])
    p = orc64.Params(seed=77, equil_cap=w.equil_cap, sweeps_per_real=5, M=6)
    res = orc64.run(z, m, T, p)
    ctx = mpr.Mpr64(_dev(torch, z), _dev(torch, m))
    ctx.set_params(T, seed=77, equil_cap=w.equil_cap, sweeps_per_real=5, M=6).equilibrate()
    st = ctx.get_stats()
    assert st.equil_sweeps == res["stats"]["sweeps"] and st.a == pytest.approx(res["stats"]["a"], rel=1e-12)
    ctx.simulate()
    pred = ctx.predict().cpu().numpy()
    free = m == 0
    assert np.array_equal(pred[~free], z[~free])
    rng_z = float(z[m == 1].max() - z[m == 1].min())
    assert np.abs(pred - res["pred"])[free].max() < 1e-9 * rng_z
    assert ctx.energy() == pytest.approx(res["stats"]["e_final"], abs=1e-12)
    st = ctx.get_stats()
    assert st.realizations == 6 and st.t == res["stats"]["t_end"]
    # spread of the realizations
    phi, zmin, zmax = orc64.transform(z, m, 77)
    eq = orc64.equilibrate(phi, m, T, p)
    acc, acc2, _ = orc64.simulate_stats(phi, m, T, eq["a"], p, t0=eq["t"])
    std_o = orc64.predict_std(acc, acc2, p.M, m, zmin, zmax)
    std_g = ctx.predict_std().cpu().numpy()
    assert np.abs(std_g - std_o)[free].max() < 1e-7 * rng_z and np.all(std_g[~free] == 0.0)
    ctx.close()


@pytest.mark.parametrize("rows,cols", [(64, 64), (150, 201), (37, 53), (2, 9), (300, 130), (65, 2)])
@pytest.mark.parametrize("q,or_mode", [(0.5, 0), (0.5, 1), (0.3, 0), (0.5, 2)])
def test_t2_tile_pass_several_sweeps_per_launch(torch_cuda, mpr, orc64, rows, cols, q, or_mode):
    """mpr64_sweep without the accepted count runs the shared-memory tile pass (k64_tilepass: up to 4 sweeps per launch on
    a frame with a halo of 8, colour planes loaded by TMA, every sweep its own Philox block): n = 1 ... 9 sweeps per call
    (passes of 4, 4 + 1, 4 + 3, 4 + 4 + 1 sweeps, from even and odd sweep indices) against n oracle sweeps, at EVERY
    prediction site within 1e-11 rad -- one and several tiles, ragged edges, odd widths (the planes' pad column)."""
    torch = torch_cuda
    if or_mode == 1 and q != 0.5:
        pytest.skip("Eq. 6 as printed is q = 1/2 only")
    z, m = _field(rows, cols, 5.0, 0.55, 900 + rows + cols)
    z = z.astype(np.float64)
    q = float(np.float32(q))               # mpr_params.q is a float field; the double path computes with its double value (R27)
    seed, T = 77, 0.03
    phi, _, _ = orc64.transform(z, m, seed)
    ctx = mpr.Mpr64(_dev(torch, z), _dev(torch, m))
    ctx.set_params(T, seed=seed, q=q, or_mode=or_mode)
    t = 0
    tol = 1e-8 if or_mode == 1 else 1e-11          # Eq. 6 as printed: atan2 of nearly cancelling q-less sums (hot state)
    for n, a in ((1, 1.0), (4, 1.5), (5, 3.0), (7, 6.0), (9, 12.0), (2, 20.0), (3, 20.0)):
        ctx.set_angles(torch.from_numpy(phi).cuda())
        ctx.set_sweep_index(t)
        assert ctx.sweep(n, a) is None
        for k in range(n):
            orc64.sweep(phi, m, q, T, a, seed, 0, t + k, or_mode)
        t += n
        got = ctx.get_angles().cpu().numpy()
        assert ctx.get_stats().t == t
        assert np.array_equal(got[m == 1], phi[m == 1])
        assert np.abs(got - phi).max() < tol, (n, a, float(np.abs(got - phi).max()))
    ctx.close()


@pytest.mark.parametrize("cap,n_fit,n_f", [(21, 20, 5), (40, 20, 7), (300, 256, 7), (300, 20, 7), (23, 20, 5)])
def test_equilibration_windows_not_aligned_with_the_check_interval(torch_cuda, mpr, orc64, cap, n_fit, n_f):
    """Alg. 2 step 5 with n_fit not a multiple of n_f (L201: the slope is checked at i >= n_fit, i % n_f == 0): the run
    stops right after the check that finds k >= 0 -- no sweep is enqueued past it (the host polls on the controller's
    schedule and a sweep after the stop does nothing) -- so t = equil_sweeps, and in double the chain is the oracle's:
    same stopping sweep, same a, same state."""
    torch = torch_cuda
    w = synth.make_workload("cfg1")
    z, m, T = w.truth[0].astype(np.float64), w.mask[0], float(w.T[0])
    ctx = mpr.Mpr64(_dev(torch, z), _dev(torch, m))
    ctx.set_params(T, seed=31, equil_cap=cap, n_fit=n_fit, n_f=n_f).equilibrate()
    st = ctx.get_stats()
    p = orc64.Params(seed=31, equil_cap=cap, n_fit=n_fit, n_f=n_f)
    phi, _, _ = orc64.transform(z, m, 31)
    eq = orc64.equilibrate(phi, m, T, p)
    assert st.equilibrated and st.t == st.equil_sweeps == eq["sweeps"]
    assert st.a == pytest.approx(eq["a"], rel=1e-12)
    assert np.abs(ctx.get_angles().cpu().numpy() - phi).max() < 1e-9
    # the next sweep draws from sweep index t on both sides
    n_acc = ctx.sweep(1, st.a, count=True)
    assert n_acc == orc64.sweep(phi, m, 0.5, T, eq["a"], 31, 0, eq["t"])
    assert np.abs(ctx.get_angles().cpu().numpy() - phi).max() < 1e-9
    ctx.close()


def test_double_and_float_paths_give_the_same_validation_measures(torch_cuda, mpr):
    """The paper's Table 2 against Table 3 (L305-321): MAE and RMSE of the double- and single-precision runs agree to
    well under the seed-to-seed noise (cfg2 shape, M = 100, s = 10; means over 4 seeds, within 1 %)."""
    torch = torch_cuda
    w = synth.make_workload("cfg2")
    z32, m, T = w.truth[0], w.mask[0], float(w.T[0])
    z64 = z32.astype(np.float64)
    c32 = mpr.Mpr(_dev(torch, z32), _dev(torch, m)); c64 = mpr.Mpr64(_dev(torch, z64), _dev(torch, m))
    rows = []
    for seed in range(8100, 8104):
        kw = dict(seed=seed, equil_cap=w.equil_cap, sweeps_per_real=10, M=100)
        c32.set_params(T, **kw).equilibrate().simulate()
        c64.set_params(T, **kw).equilibrate().simulate()
        v32 = synth.validation_measures(z32, c32.predict().cpu().numpy()[0], m)
        v64 = synth.validation_measures(z64, c64.predict().cpu().numpy(), m)
        rows.append((v32["mae"], v64["mae"], v32["rmse"], v64["rmse"]))
    c32.close(); c64.close()
    r = np.array(rows).mean(axis=0)
    assert r[0] == pytest.approx(r[1], rel=0.01) and r[2] == pytest.approx(r[3], rel=0.01)


def test_error_statuses(torch_cuda, mpr):
    torch = torch_cuda
    z, m = _field(16, 16, 3.0, 0.5, 5)
    with pytest.raises(mpr.MprError) as e:
        mpr.Mpr64(_dev(torch, z), _dev(torch, np.zeros_like(m)))
    assert e.value.name == "MPR_ERR_NO_SAMPLES"
    with pytest.raises(mpr.MprError) as e:
        mpr.Mpr64(_dev(torch, z), _dev(torch, np.ones_like(m)))
    assert e.value.name == "MPR_ERR_NO_FREE"
    with pytest.raises(mpr.MprError) as e:
        mpr.Mpr64(_dev(torch, np.full_like(z, 3.0)), _dev(torch, m))
    assert e.value.name == "MPR_ERR_DEGENERATE_RANGE"
    zz = z.copy(); zz[m == 1] = np.where(np.arange((m == 1).sum()) == 0, np.nan, zz[m == 1])
    with pytest.raises(mpr.MprError) as e:
        mpr.Mpr64(_dev(torch, zz), _dev(torch, m))
    assert e.value.name == "MPR_ERR_NONFINITE"
    ctx = mpr.Mpr64(_dev(torch, z), _dev(torch, m))
    with pytest.raises(mpr.MprError) as e:
        ctx.equilibrate()
    assert e.value.name == "MPR_ERR_STATE"
    with pytest.raises(mpr.MprError) as e:
        ctx.set_params(-1.0)
    assert e.value.name == "MPR_ERR_ARG"
    ctx.set_params(0.1, M=1)
    ctx.simulate()
    with pytest.raises(mpr.MprError) as e:
        ctx.predict_std()
    assert e.value.name == "MPR_ERR_STATE"
    ctx.close()


def test_t2_full_size_cfg4_and_cfg3_one_sweep(torch_cuda, mpr, orc64):
    """BASELINE configs[3] (4096 x 4096, 33 % removed) and configs[2] (1024 x 1024 with 64 x 64 holes) at full size, in
    the launch configuration bench.py's double_precision key times.  Generator-made near-equilibrium states (the truth
    field's own angles plus thermal-size noise at the prediction sites), as in the fp32 test of the same sizes."""
    torch = torch_cuda
    for name, a in (("cfg4", 40.0), ("cfg3", 6.0)):
        w = synth.make_workload(name)
        z, m, T = w.truth[0].astype(np.float64), w.mask[0], float(w.T[0])
        zmin, zmax, _ = orc64.minmax(z, m)
        rng = np.random.default_rng(8)
        phi = ((z - zmin) / (zmax - zmin) * TWO_PI + math.sqrt(T) * rng.standard_normal(z.shape)).clip(0.0, TWO_PI)
        ref0, _, _ = orc64.transform(z, m, w.seed)
        phi[m == 1] = ref0[m == 1]
        ctx = mpr.Mpr64(_dev(torch, z), _dev(torch, m))
        ctx.set_params(T, seed=w.seed)
        _one_sweep(orc64, ctx, phi, m, 0.5, T, a, w.seed, 123, 0)
        ctx.close()


def test_t2_one_sweep_on_a_grid_whose_state_passes_4_GiB(torch_cuda, mpr, orc64):
    """16384 x 20480 = 335 M sites: the double2 state is 5.4 GB, so byte offsets pass 2^32.  An analytic smooth field
    plus noise, 33 % removed, a near-equilibrium state; one sweep against the oracle's double build over the whole grid."""
    torch = torch_cuda
    import psutil
    if torch.cuda.get_device_properties(0).total_memory < 40 * 2 ** 30 or psutil.virtual_memory().available < 32 * 2 ** 30:
        pytest.skip("needs 25 GB of device memory and 20 GB of host memory")
    rows, cols = 16384, 20480
    rng = np.random.default_rng(6)
    r = np.arange(rows, dtype=np.float64)[:, None]; c = np.arange(cols, dtype=np.float64)[None, :]
    z = np.sin(r / 97.0) + np.cos(c / 131.0)
    z += 0.05 * rng.standard_normal(z.shape)
    m = (rng.random(z.shape, dtype=np.float32) >= 0.33).astype(np.uint8)
    T, a, seed = 2e-3, 12.0, 4243
    zmin, zmax, _ = orc64.minmax(z, m)
    phi = (z - zmin) * (TWO_PI / (zmax - zmin))
    phi += math.sqrt(T) * rng.standard_normal(z.shape)
    np.clip(phi, 0.0, TWO_PI, out=phi)
    ref0, _, _ = orc64.transform(z, m, seed)
    phi[m == 1] = ref0[m == 1]
    del ref0
    ctx = mpr.Mpr64(_dev(torch, z), _dev(torch, m))
    ctx.set_params(T, seed=seed)
    _one_sweep(orc64, ctx, phi, m, 0.5, T, a, seed, 8, 0)
    ctx.close()
