"""CPU-side checks of the boundary: the C-ABI library builds for sm_100a,
loads, exports every symbol include/mpr.h declares, and its host-only logic
(argument validation, workspace sizing, defaults) behaves as the header says.
No compute call is made: there is no GPU here."""
import ctypes as C
import os
import re

import pytest

from paper_1811_01604_b200 import build as mpr_build
from paper_1811_01604_b200 import mpr

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    mpr_build.build()
    return mpr.lib()


def _declared_symbols():
    text = open(os.path.join(ROOT, "include", "mpr.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(mpr(?:64)?_[a-z_]+)\s*\(", text)))


def test_every_declared_symbol_is_exported(lib):
    names = _declared_symbols()
    assert len(names) >= 19
    for n in names:
        assert hasattr(lib, n), n
    assert sorted(mpr.EXPORTS) == names


def test_defaults_are_reading_r7(lib):
    p = mpr.default_params()
    assert p.struct_size == C.sizeof(mpr.mpr_params)
    assert (p.q, p.n_f, p.n_fit, p.equil_cap, p.M, p.sweeps_per_real) == (0.5, 5, 20, 500, 100, 1)
    assert p.A_targ == pytest.approx(0.3) and p.k_a == 3.0 and p.or_mode == 0 and p.a_eq_mode == 0


def test_workspace_query_validates_and_scales(lib):
    for bad in [(0, 8, 8), (1, 1, 8), (1, 8, 1), (1, 70000, 8), (1, 65000, 65000)]:
        with pytest.raises(mpr.MprError) as e:
            mpr.mpr_query_workspace(*bad)
        assert e.value.name == "MPR_ERR_ARG"
    small = mpr.mpr_query_workspace(1, 64, 64)
    big = mpr.mpr_query_workspace(1, 4096, 4096)
    batch = mpr.mpr_query_workspace(32, 2048, 2048)
    assert small < 1 << 20
    # about 35.3 bytes per site: 16 (two buffers of unit vectors) + 4 + 4 (values, angles) + 4 + 4 (sum and squared
    # deviations over the realizations) + 1/8 (bitmask) + 3.2 (tile-frame entries, 2 bytes each, worst case) + padding
    assert 33 * 4096 ** 2 < big < 38 * 4096 ** 2
    assert 33 * 32 * 2048 ** 2 < batch < 38 * 32 * 2048 ** 2
    assert mpr.mpr_query_workspace(3, 37, 53) % 256 == 0
    # chains (reading R25): every further chain adds its vectors and accumulators, 24 bytes per site, nothing else
    # (the tile shape, and with it the size of the tile lists, follows the number of chains)
    one = mpr.mpr_query_workspace_chains(1, 1, 1024, 1024)
    assert one == mpr.mpr_query_workspace(1, 1024, 1024)
    four = mpr.mpr_query_workspace_chains(1, 4, 1024, 1024)
    assert 3 * 23.5 * 1024 ** 2 < four - one < 3 * 24.5 * 1024 ** 2
    for bad in [(1, 0, 8, 8), (2, 40000, 8, 8), (0, 2, 8, 8)]:
        with pytest.raises(mpr.MprError) as e:
            mpr.mpr_query_workspace_chains(*bad)
        assert e.value.name == "MPR_ERR_ARG"


def test_null_and_misuse_are_errors_not_crashes(lib):
    ctx = C.c_void_p()
    assert lib.mpr_create(C.byref(ctx), 1, 8, 8, None, None, None, 0, None) == 1          # MPR_ERR_ARG
    assert lib.mpr_create(None, 1, 8, 8, None, None, None, 0, None) == 1
    assert lib.mpr_equilibrate(None) == 1 and lib.mpr_simulate(None) == 1 and lib.mpr_predict(None, None) == 1
    assert lib.mpr_destroy(None) == 1
    assert lib.mpr_query_workspace(1, 8, 8, None) == 1
    assert ctx.value is None


def test_status_strings(lib):
    seen = set()
    for code in range(12):
        s = lib.mpr_status_string(code).decode()
        assert s and s != "unknown status"
        seen.add(s)
    assert len(seen) == 12 and set(mpr.STATUS_NAMES) == set(range(12))
    assert lib.mpr_status_string(99).decode() == "unknown status"


def test_no_cpu_fallback_in_the_product():
    """The product never imports, links or executes the oracle."""
    pkg = os.path.join(ROOT, "paper_1811_01604_b200")
    pat = re.compile(r"^\s*(from|import)\s+oracle|mpr_oracle|libmpr_oracle|orc_[a-z]", re.M)
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                assert not pat.search(open(os.path.join(dirpath, f)).read()), f


def test_infer_temperature_is_host_arithmetic_and_matches_the_oracle(lib, orc):
    """mpr_infer_temperature (Alg. 2 step 4.2, L111) needs no device: same ladders as the oracle's pins."""
    cases = [([0.01, 0.02, 0.04, 0.08], [-1 + T / 4 for T in (0.01, 0.02, 0.04, 0.08)], [-0.9975, -0.99675, -0.995, -0.9875, -0.98, -1.5, 0.3]),
             ([0.01, 0.02, 0.04, 0.08], [-0.99, -0.98, -0.95, -0.85], [-0.965, -0.99, -0.85, -0.9]),
             ([1, 2, 3, 4], [-0.99, -0.97, -0.98, -0.96], [-0.975, -0.965, -0.5])]
    for Ts, es, queries in cases:
        for e_s in queries:
            assert mpr.infer_temperature(Ts, es, e_s) == pytest.approx(orc.infer_T(e_s, Ts, es), rel=1e-6)
    with pytest.raises(mpr.MprError) as e:
        mpr.infer_temperature([2, 1], [-0.9, -0.8], -0.85)          # ladder not ascending
    assert e.value.name == "MPR_ERR_ARG"


def test_default_ladder_is_host_arithmetic_and_matches_the_oracle(lib, orc):
    """mpr_default_ladder (the ladder of Alg. 2 step 4.2 when the caller has none) needs no device; the oracle builds the
    same float32 temperatures."""
    for rows, cols, e_s in ((64, 64, -0.9946), (2048, 2048, -0.99995), (37, 53, -0.9), (4096, 4096, -1.0)):
        assert mpr.default_ladder(rows, cols, e_s) == orc.default_ladder(rows, cols, e_s)
        f = (0.1, 0.9, 1.0, 7.5)
        assert mpr.default_ladder(rows, cols, e_s, f) == orc.default_ladder(rows, cols, e_s, f)
    for bad in ((1.0, 0.5), (0.0, 1.0), (-1.0, 2.0)):
        with pytest.raises(mpr.MprError) as e:
            mpr.default_ladder(8, 8, -0.99, bad)
        assert e.value.name == "MPR_ERR_ARG"


def test_batch_limits_of_the_boundary(lib):
    """include/mpr.h: batch * chains <= 65535 states, rows * cols < 2^31 per grid, rows, cols <= 65534 (host checks)."""
    assert mpr.mpr_query_workspace_chains(65535, 1, 8, 8) > 0
    assert mpr.mpr_query_workspace_chains(255, 257, 8, 8) > 0
    for bad in ((65536, 1, 8, 8), (256, 256, 8, 8), (1, 1, 46341, 46341), (1, 1, 65535, 8), (1, 1, 8, 65535)):
        with pytest.raises(mpr.MprError) as e:
            mpr.mpr_query_workspace_chains(*bad)
        assert e.value.name == "MPR_ERR_ARG"
    assert mpr.mpr_query_workspace(1, 46340, 46340) > 35 * 46340 ** 2          # just below 2^31 sites: 75 GB
