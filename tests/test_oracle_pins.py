"""Pins of the CPU oracle against what the paper and the mathematics fix.

None of these tests touches the CUDA path.  Each names the passage it pins
(PAPER.md line / equation) and the mistake it is meant to catch.
"""
import ctypes as C
import math
import os

import numpy as np
import pytest
from scipy import integrate, stats

HERE = os.path.dirname(os.path.abspath(__file__))
PI = math.pi
TWO_PI_F = float(np.float32(2.0 * math.pi))


# ---------------------------------------------------------------------------
# P1  energy, PAPER.md L87 (Eq. 2), N_GP L109
# ---------------------------------------------------------------------------
def _parse_angle(tok):
    tok = tok.strip()
    table = {"0": 0.0, "pi": PI, "2pi": 2 * PI, "pi/2": PI / 2}
    return table[tok] if tok in table else float(tok)


def _golden_energies():
    out = []
    with open(os.path.join(HERE, "golden", "hand_energies.txt")) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            name, rows, cols, ang, H = [x.strip() for x in line.split(";")]
            out.append((name, int(rows), int(cols), [_parse_angle(a) for a in ang.split()], float(H)))
    return out


@pytest.mark.parametrize("case", _golden_energies(), ids=lambda c: c[0])
def test_energy_hand_built(orc, case):
    _, rows, cols, ang, H = case
    phi = np.array(ang, dtype=np.float32).reshape(rows, cols)
    # float storage of pi perturbs each bond by < 1e-7
    assert orc.energy(phi, 0.5) == pytest.approx(H, abs=2e-6)


def test_n_bonds(orc):
    assert orc.n_bonds(2, 2) == 4
    assert orc.n_bonds(3, 3) == 12
    for L in (5, 64, 1024):
        assert orc.n_bonds(L, L) == 2 * L * (L - 1)
    assert orc.n_bonds(3, 5) == 3 * 4 + 5 * 2


def test_energy_brute_force_random(orc):
    """Eq. 2 by an explicit double loop over ordered neighbour pairs / 2."""
    rng = np.random.default_rng(7)
    phi = (rng.random((7, 5)) * 2 * PI).astype(np.float32)
    q = 0.37
    H = 0.0
    for r in range(7):
        for c in range(5):
            for dr, dc in ((1, 0), (-1, 0), (0, 1), (0, -1)):
                rr, cc = r + dr, c + dc
                if 0 <= rr < 7 and 0 <= cc < 5:
                    H -= 0.5 * math.cos(q * (float(phi[r, c]) - float(phi[rr, cc])))
    assert orc.energy(phi, q) == pytest.approx(H, abs=1e-12)


# ---------------------------------------------------------------------------
# P2  over-relaxation, PAPER.md L156-160 (Eq. 6), L265 ("local energy
# contribution remains unchanged")
# ---------------------------------------------------------------------------
def _direct_local_energy(phi, nbrs, q):
    return -sum(math.cos(q * (phi - pj)) for pj in nbrs)


def test_or_worked_example(orc):
    q, phi, nbrs = 0.5, 1.0, (0.0, PI / 2, PI / 2)
    Cs = sum(math.cos(q * p) for p in nbrs)
    Ss = sum(math.sin(q * p) for p in nbrs)
    # closed form: C = 1 + sqrt 2, S = sqrt 2
    assert Cs == pytest.approx(1 + math.sqrt(2), abs=1e-15)
    theta = math.atan2(math.sqrt(2), 1 + math.sqrt(2))
    p1, kept, _ = orc.or_reflect(phi, Cs, Ss, q)
    assert not kept
    assert p1 == pytest.approx(4 * theta - 1.0, abs=1e-14)
    assert p1 == pytest.approx(1.1196111590, abs=1e-9)
    e0 = _direct_local_energy(phi, nbrs, q)
    e1 = _direct_local_energy(p1, nbrs, q)
    assert e0 == pytest.approx(-2.7966818219, abs=1e-9)
    assert e1 == pytest.approx(e0, abs=1e-12)
    # Eq. 6 as printed (no q inside the sums) does NOT conserve the q=1/2 energy
    C1 = sum(math.cos(p) for p in nbrs)
    S1 = sum(math.sin(p) for p in nbrs)
    p_lit, _, _ = orc.or_reflect(phi, Cs, Ss, q, mode=1, C1=C1, S1=S1)
    assert p_lit == pytest.approx(2 * math.atan2(S1, C1) - 1.0, abs=1e-14)
    assert abs(_direct_local_energy(p_lit, nbrs, q) - e0) > 1e-3


@pytest.mark.parametrize("n_nbrs", [2, 3, 4])
def test_or_conserves_local_energy_and_is_involution(orc, n_nbrs):
    rng = np.random.default_rng(100 + n_nbrs)
    n_ref = 0
    for q in (0.5, 0.3):
        for _ in range(4000):
            centre = rng.random() * 2 * PI
            spread = rng.choice([0.05, 0.5, 3.0])
            nbrs = np.clip(centre + spread * rng.standard_normal(n_nbrs), 0, 2 * PI)
            phi = float(np.clip(centre + spread * rng.standard_normal(), 0, 2 * PI))
            Cs = float(np.sum(np.cos(q * nbrs)))
            Ss = float(np.sum(np.sin(q * nbrs)))
            p1, kept, raw = orc.or_reflect(phi, Cs, Ss, q)
            assert 0.0 <= p1 <= TWO_PI_F
            if kept:
                assert p1 == phi and (raw < 0 or raw > TWO_PI_F)
                continue
            n_ref += 1
            e0 = _direct_local_energy(phi, nbrs, q)
            e1 = _direct_local_energy(p1, nbrs, q)
            assert abs(e1 - e0) <= 1e-6          # north_star tolerance
            assert abs(e1 - e0) <= 1e-12         # what double actually gives
            p2, kept2, _ = orc.or_reflect(p1, Cs, Ss, q)
            assert not kept2 or abs(p1 - TWO_PI_F) < 1e-9 or p1 < 1e-9
            if not kept2:
                assert p2 == pytest.approx(phi, abs=1e-12)
    assert n_ref > 5000


def test_or_zero_field_keeps_spin(orc):
    """atan2(0,0) = 0 -> phi' = -phi: out of range unless phi = 0 (reading R17)."""
    p1, kept, _ = orc.or_reflect(2.0, 0.0, 0.0, 0.5)
    assert kept and p1 == 2.0
    p1, kept, _ = orc.or_reflect(0.0, 0.0, 0.0, 0.5)
    assert p1 == 0.0


# ---------------------------------------------------------------------------
# P5 / P6  Philox4x32-10 and the uniform mapping
# ---------------------------------------------------------------------------
def _curand_host_words(seed, n_words):
    path = None
    for cand in ("/usr/local/cuda/lib64/libcurand.so", "libcurand.so", "libcurand.so.10"):
        try:
            lib = C.CDLL(cand)
            path = cand
            break
        except OSError:
            continue
    if path is None:
        pytest.skip("libcurand not found")
    gen = C.c_void_p()
    CURAND_RNG_PSEUDO_PHILOX4_32_10 = 161
    assert lib.curandCreateGeneratorHost(C.byref(gen), CURAND_RNG_PSEUDO_PHILOX4_32_10) == 0
    lib.curandSetPseudoRandomGeneratorSeed.argtypes = [C.c_void_p, C.c_ulonglong]
    assert lib.curandSetPseudoRandomGeneratorSeed(gen, seed) == 0
    buf = np.zeros(n_words, dtype=np.uint32)
    lib.curandGenerate.argtypes = [C.c_void_p, C.c_void_p, C.c_size_t]
    assert lib.curandGenerate(gen, buf.ctypes.data, n_words) == 0
    lib.curandDestroyGenerator.argtypes = [C.c_void_p]
    lib.curandDestroyGenerator(gen)
    return buf


@pytest.mark.parametrize("seed", [0, 1, 0x0123456789ABCDEF, 2**64 - 1])
def test_philox_matches_curand_host_generator(orc, seed):
    """cuRAND's host Philox4_32_10 generator (the one the paper used, L267):
    its n-th output quad is Philox4x32-10(counter=(0,0,n,0), key=seed)."""
    words = _curand_host_words(seed, 64)
    key = [seed & 0xFFFFFFFF, seed >> 32]
    for n in range(16):
        mine = orc.philox4x32_10([0, 0, n, 0], key)
        assert [int(x) for x in mine] == [int(x) for x in words[4 * n: 4 * n + 4]]


def test_philox_counter_words_all_matter(orc):
    base = orc.philox4x32_10([1, 2, 3, 4], [5, 6])
    for pos in range(4):
        c = [1, 2, 3, 4]
        c[pos] += 1
        assert not np.array_equal(orc.philox4x32_10(c, [5, 6]), base)
    assert not np.array_equal(orc.philox4x32_10([1, 2, 3, 4], [6, 6]), base)
    assert not np.array_equal(orc.philox4x32_10([1, 2, 3, 4], [5, 7]), base)


def test_uniform_mapping_lattice(orc):
    for x in (0, 1, 511, 512, 0x7FFFFFFF, 0x80000000, 0xFFFFFFFF, 123456789):
        u = orc.u01(x)
        assert 0.0 < u < 1.0
        assert float(np.float32(u)) == u                     # exact in float
        assert u * 2**24 == 2 * (x >> 9) + 1                 # odd numerator / 2^24
        assert orc.u01(0xFFFFFFFF - x) == pytest.approx(1.0 - u, abs=0)   # symmetric about 1/2
    assert orc.u01(0) == 2.0**-24 and orc.u01(0xFFFFFFFF) == 1.0 - 2.0**-24
    rng = np.random.default_rng(3)
    xs = rng.integers(0, 2**32, size=20000, dtype=np.uint64)
    us = np.array([orc.u01(int(x)) for x in xs])
    assert abs(us.mean() - 0.5) < 3 * math.sqrt(1 / 12 / us.size)


# ---------------------------------------------------------------------------
# P8  transform, PAPER.md L79-81 (Eq. 1)
# ---------------------------------------------------------------------------
def test_transform_endpoints_and_dyadic(orc):
    assert orc.eq1(3.0, 3.0, 11.0) == 0.0
    top = orc.eq1(11.0, 3.0, 11.0)
    assert top <= np.float32(TWO_PI_F)
    assert abs(float(top) - TWO_PI_F) <= float(np.spacing(np.float32(TWO_PI_F)))
    # zmin = 0, zmax = 1: scale = TWO_PI_F exactly, power-of-two z scale exactly
    for z in (0.0, 0.25, 0.5, 1.0):
        assert float(orc.eq1(z, 0.0, 1.0)) == z * TWO_PI_F
    # values outside the sample range cannot occur at sample sites, but the clamp holds
    assert orc.eq1(-1.0, 0.0, 1.0) == 0.0 and float(orc.eq1(2.0, 0.0, 1.0)) == TWO_PI_F


def test_transform_matches_float64_formula_and_affine_invariance(orc):
    rng = np.random.default_rng(11)
    z = rng.integers(-50, 50, size=(16, 16)).astype(np.float32)
    mask = (rng.random((16, 16)) < 0.6).astype(np.uint8)
    phi, zmin, zmax = orc.transform(z, mask, seed=5)
    m = mask.astype(bool)
    assert zmin == z[m].min() and zmax == z[m].max()
    ref = 2 * PI * (z.astype(np.float64) - float(zmin)) / (float(zmax) - float(zmin))
    assert np.max(np.abs(phi[m].astype(np.float64) - ref[m])) < 2e-6
    assert phi[m].min() == 0.0 and phi[m].max() == np.float32(TWO_PI_F)
    # Eq. 1 is invariant under z -> 4 z + 8 (exact in float for small integers)
    phi2, _, _ = orc.transform(4 * z + 8, mask, seed=5)
    assert np.array_equal(phi2[m], phi[m])
    # prediction sites: U(0, 2 pi) from the INIT stream, inside the state space
    f = ~m
    assert np.all(phi[f] > 0) and np.all(phi[f] < TWO_PI_F)
    assert np.array_equal(phi2[f], phi[f])      # INIT stream does not depend on the data


def test_init_stream_is_uniform(orc):
    z = np.zeros((128, 128), dtype=np.float32)
    z[0, 0], z[0, 1] = 0.0, 1.0
    mask = np.zeros((128, 128), dtype=np.uint8)
    mask[0, 0] = mask[0, 1] = 1
    phi, _, _ = orc.transform(z, mask, seed=99)
    f = phi[mask == 0].astype(np.float64) / TWO_PI_F
    assert abs(f.mean() - 0.5) < 4 * math.sqrt(1 / 12 / f.size)
    hist, _ = np.histogram(f, bins=16, range=(0, 1))
    chi2 = np.sum((hist - f.size / 16) ** 2 / (f.size / 16))
    assert stats.chi2.sf(chi2, 15) > 1e-3
    phi_b, _, _ = orc.transform(z, mask, seed=99, g=1)
    assert not np.array_equal(phi_b, phi)          # grid index enters the counter


# ---------------------------------------------------------------------------
# P3  sample sites fixed
# ---------------------------------------------------------------------------
def test_sample_sites_unchanged_bit_for_bit(orc):
    rng = np.random.default_rng(21)
    z = rng.standard_normal((24, 31)).astype(np.float32)
    mask = (rng.random((24, 31)) < 0.5).astype(np.uint8)
    phi, _, _ = orc.transform(z, mask, seed=1)
    before = phi.copy()
    for t in range(25):
        orc.sweep(phi, mask, 0.5, 0.05, 1.0 + t / 3, 1, 0, t)
    m = mask.astype(bool)
    assert np.array_equal(phi[m].view(np.uint32), before[m].view(np.uint32))
    assert not np.array_equal(phi[~m], before[~m])
    assert phi.min() >= 0.0 and phi.max() <= np.float32(TWO_PI_F)


# ---------------------------------------------------------------------------
# P4  Metropolis + over-relaxation sample the Gibbs density
# (Eq. 3), Alg. 1.  Histogram of a thinned chain vs numerical integration.
# ---------------------------------------------------------------------------
def _chain_one_free_site(orc, nbr_up, nbr_down, nbr_left, nbr_right, T, a, or_mode, n_keep, thin, seed):
    phi = np.zeros((3, 3), dtype=np.float32)
    # distinct junk on the diagonals: a mis-indexed neighbour would change the density
    phi[0, 0], phi[0, 2], phi[2, 0], phi[2, 2] = 0.3, 5.9, 4.4, 2.2
    phi[0, 1], phi[2, 1], phi[1, 0], phi[1, 2] = nbr_up, nbr_down, nbr_left, nbr_right
    phi[1, 1] = 3.0
    mask = np.ones((3, 3), dtype=np.uint8)
    mask[1, 1] = 0
    out = np.empty(n_keep)
    t = 0
    for i in range(n_keep):
        for _ in range(thin):
            orc.sweep(phi, mask, 0.5, T, a, seed, 0, t, or_mode)
            t += 1
        out[i] = phi[1, 1]
    return out


def _boltzmann_bin_probs(nbrs, T, q, edges):
    dens = lambda p: math.exp(sum(math.cos(q * (p - pj)) for pj in nbrs) / T)
    Z = integrate.quad(dens, 0, TWO_PI_F, epsabs=1e-12, epsrel=1e-12)[0]
    return np.array([integrate.quad(dens, edges[i], edges[i + 1], epsabs=1e-13, epsrel=1e-12)[0] / Z
                     for i in range(len(edges) - 1)])


@pytest.mark.parametrize("a", [1.0, 4.0, 37.5])
def test_proposal_is_u_scaled_by_two_pi_over_a(orc, a):
    """Alg. 1 line 3: phi'' = phi' + alpha (u - 0.5) with alpha = 2 pi / a (L156), u the FIRST of the
    site's two uniforms (the second, r, decides acceptance, line 6).  A symmetric proposal of any width has the same
    stationary law, so the chi-square pins cannot see a wrong width; this one does.  One free site, over-relaxation
    off (phi' = phi), T so high that every proposal is accepted (AP = exp(-dH/T) > 1 - 2^-24 >= r): the step of every
    sweep must be exactly 2 pi (u - 0.5) / a with u rebuilt here from the Philox words (pinned against cuRAND above),
    up to the one rounding of the state to float32."""
    seed, site, T = 777, 4, 1e12
    phi = np.full((3, 3), 3.0, dtype=np.float32)
    mask = np.ones((3, 3), dtype=np.uint8); mask[1, 1] = 0
    key = [seed & 0xFFFFFFFF, seed >> 32]
    steps = []
    for t in range(400):
        before = float(phi[1, 1])
        assert orc.sweep(phi, mask, 0.5, T, a, seed, 0, t, 2) == 1            # accepted
        x = orc.philox4x32_10([site, t >> 1, 2, 0], key)
        u = orc.u01(int(x[2 * (t & 1)]))
        want = before + TWO_PI_F * (u - 0.5) / a             # "2 pi" is the float nearest 2 pi everywhere (reading R4)
        want = want + TWO_PI_F if want < 0.0 else want - TWO_PI_F if want >= TWO_PI_F else want
        assert float(phi[1, 1]) == pytest.approx(want, abs=2.5e-7), (t, u)      # half an ulp of a float in [4, 8)
        steps.append(2.0 * PI * (u - 0.5) / a)
    steps = np.abs(np.array(steps))
    assert steps.max() <= PI / a and steps.max() >= 0.97 * PI / a              # the window is [-pi/a, pi/a], and it is used
    assert np.mean(steps) == pytest.approx(0.5 * PI / a, rel=0.1)


@pytest.mark.parametrize("nbrs,or_mode", [
    ((1.0, 2.5, 4.0, 5.5), 0),
    ((1.0, 2.5, 4.0, 5.5), 2),
    ((0.3, 0.5, 5.9, 1.0), 0),     # many rejected reflections
    ((3.0, 3.0, 3.0, 3.0), 0),
])
def test_single_site_chain_matches_boltzmann(orc, nbrs, or_mode):
    T, q = 0.5, 0.5
    samples = _chain_one_free_site(orc, *nbrs, T=T, a=1.0, or_mode=or_mode,
                                   n_keep=20000, thin=8, seed=77)
    edges = np.linspace(0, TWO_PI_F, 33)
    hist, _ = np.histogram(samples, bins=edges)
    p = _boltzmann_bin_probs(nbrs, T, q, edges)
    assert p.sum() == pytest.approx(1.0, abs=1e-9)
    expected = p * samples.size
    keep = expected > 5
    chi2 = np.sum((hist[keep] - expected[keep]) ** 2 / expected[keep])
    pval = stats.chi2.sf(chi2, keep.sum() - 1)
    assert pval > 0.01, (chi2, pval)


def test_single_site_chain_wrong_sign_would_fail(orc):
    """Power check of the chi-square pin: the density with the sign of H
    flipped is rejected by the same statistic."""
    nbrs, T, q = (1.0, 2.5, 4.0, 5.5), 0.5, 0.5
    samples = _chain_one_free_site(orc, *nbrs, T=T, a=1.0, or_mode=0, n_keep=5000, thin=8, seed=78)
    edges = np.linspace(0, TWO_PI_F, 33)
    hist, _ = np.histogram(samples, bins=edges)
    p_wrong = _boltzmann_bin_probs(nbrs, -T, q, edges)
    expected = p_wrong * samples.size
    chi2 = np.sum((hist - expected) ** 2 / np.maximum(expected, 1e-9))
    assert stats.chi2.sf(chi2, 31) < 1e-6


def test_two_adjacent_free_sites_match_joint_boltzmann(orc):
    """Checkerboard order and conditional updates: two neighbouring free sites
    (different colours) on a 3x4 grid against a 2-D quadrature of Eq. 3."""
    T, q = 0.6, 0.5
    phi = np.array([[0.4, 1.2, 2.0, 5.0],
                    [0.9, 3.0, 3.0, 2.8],
                    [6.0, 2.1, 1.0, 0.2]], dtype=np.float32)
    mask = np.ones((3, 4), dtype=np.uint8)
    mask[1, 1] = mask[1, 2] = 0
    n1 = (float(phi[0, 1]), float(phi[2, 1]), float(phi[1, 0]))      # fixed nbrs of (1,1)
    n2 = (float(phi[0, 2]), float(phi[2, 2]), float(phi[1, 3]))      # fixed nbrs of (1,2)
    n_keep, thin = 24000, 8
    s = np.empty((n_keep, 2))
    t = 0
    for i in range(n_keep):
        for _ in range(thin):
            orc.sweep(phi, mask, q, T, 1.0, 4242, 0, t, 0)
            t += 1
        s[i] = phi[1, 1], phi[1, 2]
    nb = 6
    edges = np.linspace(0, TWO_PI_F, nb + 1)
    hist, _, _ = np.histogram2d(s[:, 0], s[:, 1], bins=[edges, edges])

    def dens(y, x):     # dblquad integrates func(y, x)
        e = -sum(math.cos(q * (x - p)) for p in n1) - sum(math.cos(q * (y - p)) for p in n2) \
            - math.cos(q * (x - y))
        return math.exp(-e / T)

    probs = np.empty((nb, nb))
    for i in range(nb):
        for j in range(nb):
            probs[i, j] = integrate.dblquad(dens, edges[i], edges[i + 1], edges[j], edges[j + 1],
                                            epsabs=1e-10, epsrel=1e-9)[0]
    probs /= probs.sum()
    expected = probs * n_keep
    keep = expected > 5
    chi2 = np.sum((hist[keep] - expected[keep]) ** 2 / expected[keep])
    pval = stats.chi2.sf(chi2, keep.sum() - 1)
    assert pval > 0.01, (chi2, pval)


# ---------------------------------------------------------------------------
# P7  slope and controller, PAPER.md L192-206 (Alg. 2 step 5), L215
# ---------------------------------------------------------------------------
def test_sg_slope_closed_forms(orc):
    j = np.arange(20, dtype=np.float64)
    assert orc.sg_slope(3.0 - 0.25 * j) == pytest.approx(-0.25, abs=1e-14)
    assert orc.sg_slope(np.full(20, 7.0)) == 0.0
    assert orc.sg_slope(j ** 2) == pytest.approx(19.0, abs=1e-12)     # OLS slope of j^2 over 0..n-1 is n-1
    rng = np.random.default_rng(5)
    e = rng.standard_normal(20)
    assert orc.sg_slope(e) == pytest.approx(np.polyfit(j, e, 1)[0], abs=1e-13)


def test_equilibration_controller_follows_algorithm_2(orc):
    from paper_1811_01604_b200 import synth
    z = synth.grf(48, 48, 6.0, "gaussian", 31)
    mask = synth.bernoulli_mask(48, 48, 0.4, 32)
    T = synth.choose_T(z, mask)
    p = orc.Params(seed=9, equil_cap=400)
    phi, _, _ = orc.transform(z, mask, p.seed)
    st = orc.equilibrate(phi, mask, T, p, history=True)
    n, e, A, a = st["sweeps"], st["e_hist"], st["A_hist"], st["a_hist"]
    assert 20 < n < 400 and st["t"] == n
    # 5.2: a(i+1) = 1 + (i+1)/k_a when A < A_targ, else unchanged (a(0) = 1)
    for i in range(n):
        want = 1.0 + (i + 1) / p.k_a if A[i + 1] < p.A_targ else a[i]
        assert a[i + 1] == want
    assert st["a"] == a[n]
    # 5.4/5.5: stops at the first check (i >= n_fit, i % n_f == 0) whose OLS slope
    # over the last n_fit energies is >= 0, recomputed here with numpy.polyfit
    stop = None
    for i in range(n):
        if i >= p.n_fit and i % p.n_f == 0:
            k = np.polyfit(np.arange(p.n_fit), e[i + 2 - p.n_fit: i + 2], 1)[0]
            if k >= 0:
                stop = i + 1
                break
    assert stop == n
    # energy decreases overall during relaxation, and every e is the Eq. 2 energy per bond
    assert e[n] < e[1] - 0.1
    assert e[n] == pytest.approx(orc.energy_per_bond(phi), abs=0)


def test_equilibration_cap(orc):
    from paper_1811_01604_b200 import synth
    z = synth.grf(32, 32, 6.0, "gaussian", 41)
    mask = synth.bernoulli_mask(32, 32, 0.4, 42)
    p = orc.Params(seed=9, equil_cap=7)
    phi, _, _ = orc.transform(z, mask, p.seed)
    st = orc.equilibrate(phi, mask, 0.02, p)
    assert st["sweeps"] == 7 and st["k"] == -1.0


# ---------------------------------------------------------------------------
# P10  unconditional low-T energy: equipartition, pins O3 + O4 jointly and the
# temperature chooser's closed form (Eq. 5)
# ---------------------------------------------------------------------------
def test_unconditional_energy_equipartition(orc):
    L, T = 32, 0.01
    phi = np.full((L, L), PI, dtype=np.float32)
    mask = np.zeros((L, L), dtype=np.uint8)
    es = []
    for t in range(2600):
        orc.sweep(phi, mask, 0.5, T, 12.0, 17, 0, t, 0)
        if t >= 600:
            es.append(orc.energy_per_bond(phi))
    want = -1.0 + (L + 1) * T / (4 * L)          # -0.997421875
    got = float(np.mean(es))
    assert (1 + got) == pytest.approx(1 + want, rel=0.02), (got, want)


# ---------------------------------------------------------------------------
# O6/O7  realizations and prediction
# ---------------------------------------------------------------------------
def test_simulate_accumulates_and_predict_back_transforms(orc):
    from paper_1811_01604_b200 import synth
    z = synth.grf(20, 20, 4.0, "gaussian", 51)
    mask = synth.bernoulli_mask(20, 20, 0.5, 52)
    p = orc.Params(seed=3, M=4, sweeps_per_real=3)
    phi, zmin, zmax = orc.transform(z, mask, p.seed)
    phi_b = phi.copy()
    acc, t_end = orc.simulate(phi, mask, 0.05, 2.0, p, t0=10)
    assert t_end == 10 + 12
    # replay by hand with the single-sweep call
    want = np.zeros_like(acc)
    t = 10
    for _ in range(4):
        for _ in range(3):
            orc.sweep(phi_b, mask, 0.5, 0.05, 2.0, 3, 0, t)
            t += 1
        want += np.where(mask == 0, phi_b.astype(np.float64), 0.0)
    assert np.array_equal(acc, want) and np.array_equal(phi, phi_b)
    pred = orc.predict(acc, 4, z, mask, zmin, zmax)
    m = mask.astype(bool)
    assert np.array_equal(pred[m].view(np.uint32), z[m].view(np.uint32))
    mean_phi = acc / 4
    ref = float(zmin) + mean_phi * (float(zmax) - float(zmin)) / (2 * PI)
    assert np.max(np.abs(pred[~m] - ref[~m])) < 1e-6 * (float(zmax) - float(zmin)) + 1e-6
    # a constant angle 2 pi maps back to zmax, 0 to zmin (inverse of Eq. 1)
    ones = np.where(mask == 0, TWO_PI_F, 0.0).astype(np.float64)
    assert np.allclose(orc.predict(ones, 1, z, mask, zmin, zmax)[~m], zmax, rtol=0, atol=1e-6)
    assert np.allclose(orc.predict(0 * ones, 1, z, mask, zmin, zmax)[~m], zmin, rtol=0, atol=1e-6)


def test_or_exact_reflection_reduces_to_eq6_at_q1(orc):
    """At q = 1 the exact reflection IS Eq. 6 as printed."""
    rng = np.random.default_rng(8)
    n = 0
    for _ in range(2000):
        nbrs = rng.random(4) * 2 * PI
        phi = rng.random() * 2 * PI
        Cs, Ss = float(np.sum(np.cos(nbrs))), float(np.sum(np.sin(nbrs)))
        p0, kept, raw = orc.or_reflect(phi, Cs, Ss, 1.0, mode=0)
        p1, _, _ = orc.or_reflect(phi, Cs, Ss, 1.0, mode=1, C1=Cs, S1=Ss)
        if not kept:
            assert p0 == pytest.approx(p1, abs=1e-12)
            n += 1
        else:   # mode 0 keeps the spin where Eq. 6 would wrap; mod 2 pi they agree
            assert (raw - p1) / TWO_PI_F == pytest.approx(round((raw - p1) / TWO_PI_F), abs=1e-9)
    assert n > 500


def test_sweep_independent_of_thread_count(orc):
    """Sites of one colour are independent given the other."""
    rng = np.random.default_rng(61)
    phi0 = (rng.random((33, 47)) * TWO_PI_F).astype(np.float32)
    mask = (rng.random((33, 47)) < 0.4).astype(np.uint8)
    nthr = orc.num_threads()
    outs = []
    for n in (1, max(2, nthr)):
        orc.set_num_threads(n)
        phi = phi0.copy()
        acc = [orc.sweep(phi, mask, 0.5, 0.1, 2.0, 5, 3, t) for t in range(3)]
        outs.append((phi, acc, orc.energy(phi)))
    orc.set_num_threads(nthr)
    assert np.array_equal(outs[0][0], outs[1][0]) and outs[0][1] == outs[1][1] and outs[0][2] == outs[1][2]


# ---------------------------------------------------------------------------
# spread of the realizations, PAPER.md L212 ("Statistics of M realizations")
# ---------------------------------------------------------------------------
def test_predict_std_closed_forms(orc):
    mask = np.array([[1, 0, 0, 0]], dtype=np.uint8)
    seqs = [[0.0, 0.0, 0.0], [1.0, 2.0, 3.0], [2.5, 2.5, 2.5], [0.0, TWO_PI_F, 0.0]]    # the realizations of 4 sites
    acc = np.array([[sum(s) for s in seqs]]); acc2 = np.array([[sum(x * x for x in s) for s in seqs]])
    zmin, zmax = 10.0, 30.0
    out = orc.predict_std(acc, acc2, 3, mask, zmin, zmax)
    scale = (zmax - zmin) / TWO_PI_F
    assert out[0, 0] == 0.0                                             # a sample site: its value is data
    assert out[0, 1] == pytest.approx(1.0 * scale, rel=1e-6)            # sample s.d. of 1, 2, 3 is 1
    assert out[0, 2] == 0.0                                             # constant chain
    assert out[0, 3] == pytest.approx(math.sqrt(TWO_PI_F ** 2 * (2 / 3) / 2) * scale, rel=1e-6)
    # cancellation below zero is clamped
    assert orc.predict_std(np.array([[0.0, 3.0]]), np.array([[0.0, 3.0 - 1e-12]]), 3, mask[:, :2], 0, 1)[0, 1] == 0.0


def test_simulate_stats_sums_follow_the_chain(orc):
    """acc and acc2 are the sums of phi and phi^2 over the states after every s-th sweep of the chain."""
    rng = np.random.default_rng(12)
    z = rng.standard_normal((12, 9)).astype(np.float32)
    mask = (rng.random((12, 9)) < 0.5).astype(np.uint8); mask[0, 0] = 1; mask[-1, -1] = 0
    p = orc.Params(seed=5, M=4, sweeps_per_real=3)
    phi, _, _ = orc.transform(z, mask, p.seed)
    ref = phi.copy()
    acc, acc2, t_end = orc.simulate_stats(phi, mask, 0.2, 2.0, p, t0=7)
    s1 = np.zeros(ref.shape); s2 = np.zeros(ref.shape); t = 7
    for _ in range(p.M):
        for _ in range(p.sweeps_per_real):
            orc.sweep(ref, mask, p.q, 0.2, 2.0, p.seed, 0, t); t += 1
        s1 += ref.astype(np.float64); s2 += ref.astype(np.float64) ** 2
    free = mask == 0
    assert t_end == t and np.array_equal(ref, phi)
    assert np.array_equal(acc[free], s1[free]) and np.array_equal(acc2[free], s2[free])
    assert np.all(acc[~free] == 0) and np.all(acc2[~free] == 0)
    assert np.all(acc2[free] * p.M >= acc[free] ** 2 * (1 - 1e-12))      # Cauchy-Schwarz
    # the mean-only entry point is the same chain
    phi2, _, _ = orc.transform(z, mask, p.seed)
    acc_only, _ = orc.simulate(phi2, mask, 0.2, 2.0, p, t0=7)
    assert np.array_equal(acc_only, acc)


# ---------------------------------------------------------------------------
# chain parallelism (reading R25): the M realizations
# made by several chains forked from the equilibrated state
# ---------------------------------------------------------------------------
def test_chains_one_chain_is_step_6(orc):
    rng = np.random.default_rng(31)
    z = rng.standard_normal((10, 13)).astype(np.float32)
    mask = (rng.random((10, 13)) < 0.4).astype(np.uint8); mask[0, 0] = 1; mask[-1, -1] = 0
    p = orc.Params(seed=9, M=5, sweeps_per_real=2)
    phi, _, _ = orc.transform(z, mask, p.seed)
    start = phi.copy()
    acc, acc2, M_tot, t_end, finals = orc.simulate_chains(start, mask, 0.3, 1.5, p, chains=1, t0=4)
    a1, a2, t1 = orc.simulate_stats(phi, mask, 0.3, 1.5, p, t0=4)
    assert M_tot == 5 and t_end == t1 == 4 + 10
    assert np.array_equal(acc, a1) and np.array_equal(acc2, a2) and np.array_equal(finals[0], phi)


def test_chains_pool_the_hand_swept_realizations(orc):
    """Mean and spread of simulate_chains are numpy's mean and sample s.d. over the realizations of every chain,
    each swept by hand from a copy of the start state with the chain's own Philox grid word g + c * batch."""
    rng = np.random.default_rng(32)
    z = rng.standard_normal((9, 11)).astype(np.float32)
    mask = (rng.random((9, 11)) < 0.5).astype(np.uint8); mask[0, 0] = 1; mask[-1, -1] = 0
    p = orc.Params(seed=21, M=7, sweeps_per_real=2)           # 3 chains -> ceil(7 / 3) = 3 realizations each
    phi, zmin, zmax = orc.transform(z, mask, p.seed, g=2)
    start = phi.copy()
    acc, acc2, M_tot, t_end, finals = orc.simulate_chains(phi, mask, 0.25, 2.0, p, chains=3, g=2, batch=5, t0=6)
    assert np.array_equal(phi, start)                           # the start state is not advanced
    assert orc.chains_realizations(7, 3) == 3 and M_tot == 9 and t_end == 6 + 3 * 2
    reals = []
    for c in range(3):
        state = start.copy(); t = 6
        for _ in range(3):
            for _ in range(2):
                orc.sweep(state, mask, p.q, 0.25, 2.0, p.seed, 2 + 5 * c, t); t += 1
            reals.append(state.astype(np.float64))
        assert np.array_equal(state, finals[c])
    reals = np.stack(reals)
    free = mask == 0
    assert not np.array_equal(finals[0], finals[1])             # the chains do differ
    pred = orc.predict(acc, M_tot, z, mask, zmin, zmax)
    std = orc.predict_std(acc, acc2, M_tot, mask, zmin, zmax)
    scale = (float(zmax) - float(zmin)) / TWO_PI_F
    assert np.allclose(pred[free], float(zmin) + reals.mean(axis=0)[free] * scale, rtol=1e-6, atol=1e-6)
    assert np.allclose(std[free], reals.std(axis=0, ddof=1)[free] * scale, rtol=1e-5, atol=1e-6)


def test_chains_pooled_moments_match_boltzmann(orc):
    """One free site between four fixed neighbours: the first two moments pooled over 40 chains forked from a
    burnt-in state equal those of the Gibbs density (Eq. 3) by quadrature, within the chains' own sampling error."""
    nbrs, T, q = (1.0, 2.5, 4.0, 5.5), 0.5, 0.5
    phi = np.zeros((3, 3), dtype=np.float32)
    phi[0, 0], phi[0, 2], phi[2, 0], phi[2, 2] = 0.3, 5.9, 4.4, 2.2
    phi[0, 1], phi[2, 1], phi[1, 0], phi[1, 2] = nbrs
    phi[1, 1] = 3.0
    mask = np.ones((3, 3), dtype=np.uint8); mask[1, 1] = 0
    for t in range(50):
        orc.sweep(phi, mask, q, T, 1.0, 123, 0, t)
    p = orc.Params(seed=123, M=40 * 500, sweeps_per_real=8)
    acc, acc2, M_tot, _, _ = orc.simulate_chains(phi, mask, T, 1.0, p, chains=40, t0=50)
    dens = lambda x: math.exp(sum(math.cos(q * (x - pj)) for pj in nbrs) / T)
    Z = integrate.quad(dens, 0, TWO_PI_F, epsabs=1e-13)[0]
    m1 = integrate.quad(lambda x: x * dens(x), 0, TWO_PI_F, epsabs=1e-13)[0] / Z
    m2 = integrate.quad(lambda x: x * x * dens(x), 0, TWO_PI_F, epsabs=1e-13)[0] / Z
    m4 = integrate.quad(lambda x: x ** 4 * dens(x), 0, TWO_PI_F, epsabs=1e-13)[0] / Z
    # realizations 8 sweeps apart are nearly independent; allow 4.5 standard errors at an effective size of M / 2
    n_eff = M_tot / 2
    assert abs(acc[1, 1] / M_tot - m1) < 4.5 * math.sqrt((m2 - m1 * m1) / n_eff)
    assert abs(acc2[1, 1] / M_tot - m2) < 4.5 * math.sqrt((m4 - m2 * m2) / n_eff)


# ---------------------------------------------------------------------------
# quantiles from the first two moments of the realizations (reading R26)
# ---------------------------------------------------------------------------
def test_inverse_normal_cdf_against_scipy_and_closed_forms(orc):
    assert orc.inv_norm_cdf(0.5) == pytest.approx(0.0, abs=1e-12)
    assert orc.inv_norm_cdf(0.8413447460685429) == pytest.approx(1.0, abs=1e-10)      # Phi(1)
    assert orc.inv_norm_cdf(0.975) == pytest.approx(1.959963984540054, abs=1e-10)
    for p in (1e-9, 1e-3, 0.05, 0.3, 0.7, 0.999, 1 - 1e-9):
        assert orc.inv_norm_cdf(p) == pytest.approx(stats.norm.ppf(p), abs=1e-8)
        assert orc.inv_norm_cdf(p) == pytest.approx(-orc.inv_norm_cdf(1 - p), abs=1e-6)


def test_predict_quantile_closed_forms(orc):
    mask = np.array([[1, 0, 0, 0]], dtype=np.uint8)
    z = np.array([[17.0, np.nan, np.nan, np.nan]], dtype=np.float32)
    seqs = [[0.0] * 3, [1.0, 2.0, 3.0], [2.5, 2.5, 2.5], [0.0, TWO_PI_F, 0.0]]
    acc = np.array([[sum(s) for s in seqs]]); acc2 = np.array([[sum(x * x for x in s) for s in seqs]])
    zmin, zmax = 10.0, 30.0
    scale = (zmax - zmin) / TWO_PI_F
    med = orc.predict_quantile(acc, acc2, 3, 0.5, z, mask, zmin, zmax)
    assert med[0, 0] == np.float32(17.0)                                               # a sample site returns its datum
    assert np.array_equal(med[0, 1:], orc.predict(acc, 3, z, mask, zmin, zmax)[0, 1:]) # the median is the mean
    up = orc.predict_quantile(acc, acc2, 3, 0.8413447460685429, z, mask, zmin, zmax)
    assert up[0, 1] == pytest.approx(zmin + (2.0 + 1.0) * scale, rel=1e-6)             # mean 2, s.d. 1: one s.d. up
    assert up[0, 2] == pytest.approx(zmin + 2.5 * scale, rel=1e-6)                     # no spread: every quantile is the value
    lo = orc.predict_quantile(acc, acc2, 3, 0.001, z, mask, zmin, zmax)
    assert lo[0, 3] == np.float32(zmin)                                                # clamped to the data range
    assert orc.predict_quantile(acc, acc2, 3, 0.999, z, mask, zmin, zmax)[0, 3] == pytest.approx(zmax)
    qs = [orc.predict_quantile(acc, acc2, 3, p, z, mask, zmin, zmax)[0, 1] for p in (0.1, 0.3, 0.5, 0.7, 0.9)]
    assert all(a < b for a, b in zip(qs, qs[1:]))
    assert qs[0] + qs[4] == pytest.approx(2 * qs[2], rel=1e-6)                          # symmetric about the mean
