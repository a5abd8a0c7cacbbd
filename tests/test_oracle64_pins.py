"""Pins of the oracle built with double storage (oracle/mpr_oracle64.py: the same C source with -DORC_F64; the paper's
double-precision program, Table 2).  The algorithm is pinned by tests/test_oracle_pins.py on the
float build; these tests check what the storage type changes -- closed forms now hold to double accuracy, Eq. 1 in
double, the state space [0, 2 pi] with the double 2 pi -- and that the two builds stay the same method."""
import math
import os

import numpy as np
import pytest
from scipy import integrate, stats

from test_oracle_pins import _golden_energies, _boltzmann_bin_probs      # tests/ is on sys.path (rootdir conftest)

PI = math.pi
TWO_PI = 2.0 * math.pi


@pytest.fixture(scope="module")
def orc64():
    from oracle import mpr_oracle64
    mpr_oracle64.lib()
    assert mpr_oracle64.REAL is np.float64 and mpr_oracle64.TWO_PI_F == TWO_PI
    return mpr_oracle64


@pytest.mark.parametrize("case", _golden_energies(), ids=lambda c: c[0])
def test_energy_hand_built_to_double_accuracy(orc64, case):
    _, rows, cols, ang, H = case
    phi = np.array(ang, dtype=np.float64).reshape(rows, cols)
    assert orc64.energy(phi, 0.5) == pytest.approx(H, abs=1e-14 * max(1.0, abs(H)) * 10)


def test_or_conserves_local_energy_to_double_accuracy_through_a_sweep(orc64):
    """One free site, T -> 0 and a huge a: the Metropolis step cannot move, the sweep is the reflection alone; the
    local energy (L156 'energy conserving') is kept to 1e-13 and a second sweep returns the spin (involution)."""
    rng = np.random.default_rng(3)
    for _ in range(50):
        phi = (rng.random((3, 3)) * TWO_PI)
        phi[1, 1] = rng.random() * TWO_PI
        mask = np.ones((3, 3), dtype=np.uint8); mask[1, 1] = 0
        nb = [phi[0, 1], phi[2, 1], phi[1, 0], phi[1, 2]]
        e0 = -sum(math.cos(0.5 * (phi[1, 1] - pj)) for pj in nb)
        p0 = phi[1, 1]
        orc64.sweep(phi, mask, 0.5, 1e-300, 1e12, 1, 0, 0)
        e1 = -sum(math.cos(0.5 * (phi[1, 1] - pj)) for pj in nb)
        assert abs(e1 - e0) < 1e-13 + 4e-12            # + the proposal's 2 pi / a (1e12) displacement times dE/dphi
        moved = abs(phi[1, 1] - p0) > 1e-9
        orc64.sweep(phi, mask, 0.5, 1e-300, 1e12, 1, 0, 1)
        if moved:
            assert abs(phi[1, 1] - p0) < 1e-10


def test_transform_in_double(orc64):
    z = np.array([[1.0, 2.0, 4.0, 9.0]])
    mask = np.array([[1, 1, 0, 1]], dtype=np.uint8)
    phi, zmin, zmax = orc64.transform(z, mask, 3)
    assert (zmin, zmax) == (1.0, 9.0) and phi.dtype == np.float64
    assert phi[0, 0] == 0.0 and phi[0, 3] == pytest.approx(TWO_PI, abs=1e-15) and phi[0, 3] <= TWO_PI
    assert phi[0, 1] == (2.0 - 1.0) * (TWO_PI / 8.0)                     # the pinned operation order, in double
    assert 0.0 < phi[0, 2] < TWO_PI                                        # the free site: 2 pi u, u on the 2^-24 lattice
    u = phi[0, 2] / TWO_PI * 2 ** 24
    assert abs(u - round(u)) < 1e-6 and round(u) % 2 == 1
    rng = np.random.default_rng(5)
    z = rng.standard_normal((16, 16)); mask = (rng.random((16, 16)) < 0.5).astype(np.uint8); mask[0, 0] = 1; mask[-1, -1] = 0
    phi, zmin, zmax = orc64.transform(z, mask, 9)
    s = mask == 1
    assert np.allclose(phi[s], (z[s] - zmin) * TWO_PI / (zmax - zmin), rtol=0, atol=4e-15)


def test_fixed_sites_bit_identical_and_state_in_range(orc64):
    rng = np.random.default_rng(6)
    z = rng.standard_normal((12, 10)); mask = (rng.random((12, 10)) < 0.4).astype(np.uint8); mask[0, 0] = 1; mask[-1, -1] = 0
    phi, _, _ = orc64.transform(z, mask, 4)
    ref = phi.copy()
    for t in range(30):
        orc64.sweep(phi, mask, 0.5, 0.3, 1.0, 4, 0, t)
    assert np.array_equal(phi[mask == 1], ref[mask == 1])
    assert phi.min() >= 0.0 and phi.max() <= TWO_PI
    assert not np.array_equal(phi[mask == 0], ref[mask == 0])


def test_single_site_chain_matches_boltzmann_in_double(orc64):
    nbrs, T, q = (1.0, 2.5, 4.0, 5.5), 0.5, 0.5
    phi = np.zeros((3, 3)); phi[0, 0], phi[0, 2], phi[2, 0], phi[2, 2] = 0.3, 5.9, 4.4, 2.2
    phi[0, 1], phi[2, 1], phi[1, 0], phi[1, 2] = nbrs
    phi[1, 1] = 3.0
    mask = np.ones((3, 3), dtype=np.uint8); mask[1, 1] = 0
    out = np.empty(20000); t = 0
    for i in range(out.size):
        for _ in range(8):
            orc64.sweep(phi, mask, q, T, 1.0, 79, 0, t); t += 1
        out[i] = phi[1, 1]
    edges = np.linspace(0, TWO_PI, 33)
    hist, _ = np.histogram(out, bins=edges)
    expected = _boltzmann_bin_probs(nbrs, T, q, edges) * out.size
    chi2 = np.sum((hist - expected) ** 2 / expected)
    assert stats.chi2.sf(chi2, 31) > 0.01


def test_double_and_float_builds_are_the_same_method(orc, orc64):
    """Same field, mask, seed: the two builds' states agree to float accuracy after Eq. 1 and after one sweep, except at
    sites whose Metropolis decision was near the threshold; energies per bond agree to 1e-6."""
    rng = np.random.default_rng(8)
    z = rng.standard_normal((48, 40)); mask = (rng.random((48, 40)) < 0.5).astype(np.uint8); mask[0, 0] = 1; mask[-1, -1] = 0
    p64, _, _ = orc64.transform(z, mask, 11)
    p32, _, _ = orc.transform(z.astype(np.float32), mask, 11)
    # start both from the float state so that only the arithmetic differs
    p64 = p32.astype(np.float64)
    a32 = orc.sweep(p32, mask, 0.5, 0.05, 2.0, 11, 0, 0, diag=True)
    a64 = orc64.sweep(p64, mask, 0.5, 0.05, 2.0, 11, 0, 0)
    margin = a32[1]
    ok = (mask == 1) | (margin > 1e-4)
    assert (~ok).sum() <= 5
    # where no decision was close the two states differ by float rounding of the stored angle only
    d = np.abs(p64 - p32.astype(np.float64))
    far = ok.copy()
    # a flipped site changes its later-updated neighbours too: exclude sites next to a near-threshold one
    bad = ~ok
    near = bad.copy(); near[1:, :] |= bad[:-1, :]; near[:-1, :] |= bad[1:, :]; near[:, 1:] |= bad[:, :-1]; near[:, :-1] |= bad[:, 1:]
    assert d[~near].max() < 2e-5
    assert orc64.energy_per_bond(p64) == pytest.approx(orc.energy_per_bond(p32), abs=1e-4)
    assert abs(int(a64 if not isinstance(a64, tuple) else a64[0]) - int(a32[0])) <= 5


def test_unconditional_equipartition_in_double(orc64):
    """No fixed site, ordered start, T = 0.01, L = 32: <e> = -1 + (L + 1) T / (4 L) (reading R15), within 1 % of 1 + e."""
    L, T = 32, 0.01
    phi = np.full((L, L), PI)
    mask = np.zeros((L, L), dtype=np.uint8)
    t = 0; a = 8.0
    for _ in range(300):
        orc64.sweep(phi, mask, 0.5, T, a, 17, 0, t); t += 1
    es = []
    for _ in range(600):
        orc64.sweep(phi, mask, 0.5, T, a, 17, 0, t); t += 1
        es.append(orc64.energy_per_bond(phi))
    assert 1.0 + np.mean(es) == pytest.approx((L + 1) * T / (4 * L), rel=0.02)
