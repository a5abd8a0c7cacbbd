"""Driver for compute-sanitizer runs of the CUDA path: every kernel family once, on
small inputs, so that `compute-sanitizer --tool memcheck|racecheck|synccheck python tests/sanitizer_driver.py` ends
within minutes.  Not collected by pytest (no test_ prefix); it asserts only that the calls succeed and the results are
finite -- the findings are the sanitizer's.  Summaries of the runs are kept under profiles/.

Covered: create (min/max, transform, tile lists), set_params (initial state), the tile pass as
  - k_tilepass<EQUIL> (one-tile grid, in-pass Alg. 2 step 5),
  - k_tilepass<FUSED> K = 1 + k_controller (multi-tile equilibration),
  - the non-fused K = 4 pass with and without the short polynomials, with the PASS_ACCUMULATE tail (both walks),
  - general q, or_mode 1 and 2, chains, a batch,
energy, sample energy, measure_energy (unconditional context), predict / predict_std / predict_quantile, angle import /
export, and the double-precision path (k64_*)."""
import os
import sys

import numpy as np
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
from paper_1811_01604_b200 import mpr, synth  # noqa: E402


def field(rows, cols, ell, p, seed):
    z = synth.grf(rows, cols, ell, "gaussian", seed)
    m = synth.bernoulli_mask(rows, cols, p, seed + 1)
    m.flat[0] = 1; m.flat[-1] = 0
    return z, m


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def run_fp32(rows, cols, batch=1, chains=1, q=0.5, or_mode=0, a=None, cap=25, M=2, s=5):
    zs, ms = zip(*[field(rows, cols, 6.0, 0.45, 10 + g) for g in range(batch)])
    z, m = np.stack(zs), np.stack(ms)
    ctx = mpr.Mpr(dev(z), dev(m), chains=chains)
    T = [synth.choose_T(zs[g], ms[g], q) for g in range(batch)]
    ctx.set_params(T, seed=7, q=q, or_mode=or_mode, equil_cap=cap, M=M, sweeps_per_real=s)
    ctx.sample_energy()
    ctx.equilibrate()
    if a is not None:
        ctx.sweep(9, a)                      # K = 4, 4, 1 without the count
        ctx.sweep(3, a, count=True)
    ctx.simulate()
    out = [ctx.predict(), ctx.predict_std(), ctx.predict_quantile(0.9), ctx.get_angles()]
    ctx.set_angles(out[3])
    e = ctx.energy()
    assert all(np.isfinite(e)) and all(bool(torch.isfinite(o).all()) for o in out)
    tiling = ctx.get_tiling()
    ctx.close()
    return tiling


def main():
    if "--lib" in sys.argv:                  # e.g. the -DMPR_CHECKED build (paper_1811_01604_b200.build.build_checked())
        mpr.LIB_PATH = os.path.abspath(sys.argv[sys.argv.index("--lib") + 1])
        print("library:", mpr.LIB_PATH)
    print("one tile (in-pass equilibration):", run_fp32(64, 64, a=2.0))
    print("multi-tile, low tiles:", run_fp32(130, 150, a=3.0))
    print("multi-tile, short polynomials, width not a multiple of 4:", run_fp32(150, 131, a=30.0))
    print("64-row tiles (batch fills the device):", run_fp32(256, 256, batch=8, a=12.0, cap=22, M=2, s=4))
    print("chains:", run_fp32(96, 200, chains=3, a=2.0))
    print("general q:", run_fp32(140, 140, q=0.3, a=2.0))
    print("Eq. 6 as printed:", run_fp32(140, 140, or_mode=1, a=2.0))
    print("no over-relaxation:", run_fp32(140, 140, or_mode=2, a=25.0))
    # unconditional chains (Alg. 2 step 4.2)
    table = mpr.energy_table(140, 140, [0.01, 0.02], 5, torch.device("cuda:0"), seed=3, equil_cap=20)
    assert all(np.isfinite(table))
    print("energy table:", table)
    # the double-precision path
    z, m = field(130, 150, 6.0, 0.45, 30)
    c64 = mpr.Mpr64(dev(z.astype(np.float64)), dev(m))
    c64.set_params(synth.choose_T(z, m), seed=7, equil_cap=25, M=2, sweeps_per_real=3).equilibrate().simulate()
    out = [c64.predict(), c64.predict_std(), c64.get_angles()]
    c64.set_angles(out[2])
    c64.sweep(2, 2.0, count=True)
    assert np.isfinite(c64.energy()) and all(bool(torch.isfinite(o).all()) for o in out)
    c64.close()
    c64 = mpr.Mpr64(dev(z.astype(np.float64)), dev(m))
    c64.set_params(synth.choose_T(z, m), seed=7, M=2, sweeps_per_real=7).simulate()     # the double tile pass: 4 + 3 sweeps
    c64.sweep(9, 3.0)
    assert bool(torch.isfinite(c64.predict()).all())
    c64.close()
    print("double-precision path: ok")
    torch.cuda.synchronize()
    print("sanitizer driver: all calls returned MPR_OK")


if __name__ == "__main__":
    main()
