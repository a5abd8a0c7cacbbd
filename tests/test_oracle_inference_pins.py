"""Pins of the oracle's Alg. 2 step 4 (parameter inference) against what the
paper and the mathematics fix: closed-form sample specific energies of hand-built grids (Eq. 4), the
relation e_s = H / N_GP when every site is a sample (Eq. 2 / Eq. 5), the unconditional energy of a
2 x 2 grid against 4-D Gauss-Legendre quadrature of the Boltzmann average (Eq. 3, Eq. 5), the low-T
equipartition form of e(T, L), and the inversion on an exactly linear ladder."""
import math

import numpy as np
import pytest

PI = math.pi
TWO_PI_F = float(np.float32(2.0 * math.pi))


def test_sample_energy_hand_built(orc):
    ones = np.ones((2, 2), dtype=np.uint8)
    # every bond differs by pi: cos(pi/2) = 0
    e, n = orc.sample_energy(np.array([[0, PI], [PI, 2 * PI]], dtype=np.float32), ones)
    assert n == 4 and abs(e) < 1e-6
    # two bonds cos 0 = +1, two bonds cos(+-pi) = -1: 0 and 2 pi are opposite states
    e, n = orc.sample_energy(np.array([[0, 0], [0, TWO_PI_F]], dtype=np.float32), ones)
    assert n == 4 and abs(e) < 1e-6
    # aligned spins, centre missing: the 4 bonds of the centre do not count (N_SP = 12 - 4)
    m = np.ones((3, 3), dtype=np.uint8); m[1, 1] = 0
    phi = np.full((3, 3), 1.25, dtype=np.float32); phi[1, 1] = 5.0      # value at a non-sample site is ignored
    e, n = orc.sample_energy(phi, m)
    assert n == 8 and e == pytest.approx(-1.0, abs=1e-12)
    # phi_ij = i + j, q = 1/2: every bond differs by 1 -> e_s = -cos(1/2), whatever the mask
    phi = np.add.outer(np.arange(4), np.arange(5)).astype(np.float32)
    m = np.ones((4, 5), dtype=np.uint8); m[0, 0] = m[2, 3] = m[3, 4] = 0
    e, n = orc.sample_energy(phi, m)
    assert n == 31 - 2 - 4 - 2 and e == pytest.approx(-math.cos(0.5), abs=1e-12)
    # q enters: q = 0.25
    e, _ = orc.sample_energy(phi, m, q=0.25)
    assert e == pytest.approx(-math.cos(0.25), abs=1e-12)
    # isolated samples only: no pair
    m = np.zeros((3, 3), dtype=np.uint8); m[0, 0] = m[2, 2] = m[0, 2] = 1
    assert orc.sample_energy(phi[:3, :3].copy(), m) == (0.0, 0)


def test_sample_energy_equals_energy_per_bond_when_every_site_is_a_sample(orc):
    rng = np.random.default_rng(5)
    phi = (rng.random((17, 23)) * TWO_PI_F).astype(np.float32)
    e, n = orc.sample_energy(phi, np.ones_like(phi, dtype=np.uint8))
    assert n == orc.n_bonds(17, 23)
    assert e == pytest.approx(orc.energy_per_bond(phi), abs=1e-12)


def test_sample_energy_brute_force_on_random_mask(orc):
    rng = np.random.default_rng(6)
    phi = (rng.random((9, 11)) * TWO_PI_F).astype(np.float32)
    m = (rng.random((9, 11)) < 0.6).astype(np.uint8)
    tot, cnt = 0.0, 0
    for r in range(9):
        for c in range(11):
            for dr, dc in ((0, 1), (1, 0), (0, -1), (-1, 0)):          # Eq. 4's double sum: ordered pairs
                rr, cc = r + dr, c + dc
                if 0 <= rr < 9 and 0 <= cc < 11 and m[r, c] and m[rr, cc]:
                    tot += math.cos(0.5 * (float(phi[r, c]) - float(phi[rr, cc]))); cnt += 1
    e, n = orc.sample_energy(phi, m)
    assert 2 * n == cnt and e == pytest.approx(-tot / cnt, abs=1e-12)


def _quadrature_energy_2x2(T, q=0.5, order=24):
    """<H> / N_GP of the 2 x 2 grid with open boundaries by Gauss-Legendre quadrature over [0, 2 pi]^4."""
    x, w = np.polynomial.legendre.leggauss(order)
    x = PI * (x + 1.0); w = PI * w
    a, b, c, d = np.meshgrid(x, x, x, x, indexing="ij")              # a b / c d
    H = -(np.cos(q * (a - b)) + np.cos(q * (c - d)) + np.cos(q * (a - c)) + np.cos(q * (b - d)))
    W = np.einsum("i,j,k,l->ijkl", w, w, w, w) * np.exp(-H / T)
    return float((H * W).sum() / W.sum()) / 4.0


def test_unconditional_energy_of_the_2x2_grid_matches_quadrature(orc):
    T = 0.5
    want = _quadrature_energy_2x2(T)
    assert abs(_quadrature_energy_2x2(T, order=16) - want) < 1e-6     # the quadrature itself has converged
    phi = np.full((2, 2), PI, dtype=np.float32)
    mask = np.zeros((2, 2), dtype=np.uint8)
    es = []
    for t in range(42000):
        orc.sweep(phi, mask, 0.5, T, 1.0, 99, 0, t, 0)
        if t >= 2000:
            es.append(orc.energy_per_bond(phi))
    es = np.array(es)
    blocks = es.reshape(100, -1).mean(axis=1)
    err = blocks.std(ddof=1) / math.sqrt(len(blocks))
    assert abs(es.mean() - want) < 4.0 * err + 1e-3, (es.mean(), want, err)
    assert err < 0.01


def test_energy_table_follows_equipartition_at_low_T_and_is_monotone(orc):
    L = 32
    Ts = [0.0005, 0.004, 0.008, 0.016, 0.032]      # the lowest needs a = 20: the burn-in must not stop early
    p = orc.Params(seed=21, equil_cap=400)
    es = orc.energy_table(L, L, Ts, p, n_meas=300)
    want = [-1.0 + (L + 1) * T / (4 * L) for T in Ts]
    for got, w in zip(es, want):
        assert (1 + got) == pytest.approx(1 + w, rel=0.03), (es, want)
    assert np.all(np.diff(es) > 0)
    # chains differ by their Philox grid index: same T twice gives two different (but close) averages
    e2 = orc.energy_table(L, L, [0.016, 0.016], p, n_meas=50)
    assert e2[0] != e2[1] and (1 + e2[0]) == pytest.approx(1 + e2[1], rel=0.05)


def test_infer_T_on_ladders(orc):
    Ts = [0.01, 0.02, 0.04, 0.08]
    es = [-1 + T / 4 for T in Ts]                                    # exactly linear ladder
    for T in (0.01, 0.013, 0.02, 0.05, 0.08):
        assert orc.infer_T(-1 + T / 4, Ts, es) == pytest.approx(T, rel=1e-12)
    assert orc.infer_T(-1.5, Ts, es) == Ts[0] and orc.infer_T(0.3, Ts, es) == Ts[-1]   # outside: the nearer end
    # curved ladder: the interpolant is used, not the nearest point
    es = [-0.99, -0.98, -0.95, -0.85]
    assert orc.infer_T(-0.965, Ts, es) == pytest.approx(0.03, rel=1e-12)
    # a noisy, non-monotone ladder: the first bracketing segment
    assert orc.infer_T(-0.975, [1, 2, 3, 4], [-0.99, -0.97, -0.98, -0.96]) == pytest.approx(1.75)


def test_default_ladder_is_centred_where_the_chain_energy_meets_e_s(orc):
    """Step 4.2 without a ladder of the caller's: the oracle centres its ladder on the temperature at which the
    low-temperature equipartition energy equals e_s (reading R15).  Pinned by the chains themselves, not by the formula:
    an unconditional 32 x 32 chain run AT the centre has (1 + e) within 1 % of (1 + e_s), at the ladder's ends it has
    not (factors 1/4 and 4 give a quarter and four times the excess energy), and the default ladder is ascending
    with the standard factors."""
    L, e_s = 32, -0.9975
    centre = orc.default_ladder(L, L, e_s, (1.0,))[0]
    p = orc.Params(seed=11, equil_cap=300)
    ladder = orc.default_ladder(L, L, e_s)
    assert len(ladder) == 5 and all(b > a for a, b in zip(ladder, ladder[1:]))
    assert [t / centre for t in ladder] == pytest.approx([0.25, 0.5, 1.0, 2.0, 4.0], rel=1e-6)
    e = orc.energy_table(L, L, [ladder[0], centre, ladder[-1]], p, 400)
    assert (1 + e[1]) == pytest.approx(1 + e_s, rel=0.01)
    assert (1 + e[0]) == pytest.approx(0.25 * (1 + e_s), rel=0.02)
    assert (1 + e[2]) == pytest.approx(4.0 * (1 + e_s), rel=0.03)
    # the whole of step 4 on a full sample set drawn from such a chain returns the chain's temperature
    phi = np.full((L, L), np.float32(PI), dtype=np.float32)
    mask0 = np.zeros((L, L), dtype=np.uint8)
    a, T_true = 1.0, 0.02
    for t in range(400):
        acc = orc.sweep(phi, mask0, 0.5, T_true, a, 5, 0, t)
        if acc / (L * L) < 0.3:
            a = 1.0 + (t + 1) / 3.0
    T_hat, e_chain, Ts, table = orc.infer_T_auto(phi, np.ones((L, L), dtype=np.uint8), orc.Params(seed=12, equil_cap=300), 300)
    assert e_chain == pytest.approx(orc.energy_per_bond(phi), abs=1e-12)
    assert T_hat == pytest.approx(T_true, rel=0.1)          # one state's energy fluctuates by ~3 % at this size


def test_harness_temperature_is_the_sample_energy_through_the_closed_form(orc):
    """synth.choose_T (the input generator's temperature, reading R15) is e_s of Eq. 4 pushed through the equipartition
    line: checked against the oracle's e_s and ladder centre on three kinds of input, so that the generator cannot
    drift from the method (it is an input recipe, but it does restate Eq. 1 and Eq. 4)."""
    from paper_1811_01604_b200 import synth
    for rows, cols, ell, p_rm, seed in ((64, 64, 8.0, 0.33, 1), (40, 90, 3.0, 0.66, 2), (128, 128, 30.0, 0.5, 3)):
        z = synth.grf(rows, cols, ell, "gaussian", seed)
        m = synth.bernoulli_mask(rows, cols, p_rm, seed + 10)
        phi, _, _ = orc.transform(z, m, 0)
        e_s, n_sp = orc.sample_energy(phi, m)
        assert n_sp > 0
        T_orc = orc.default_ladder(rows, cols, e_s, (1.0,))[0]
        # Eq. 1 in float32 (oracle) against float64 (generator): (1 + e_s) ~ 1e-3 .. 1e-5 carries ~1e-4 relative
        assert synth.choose_T(z, m) == pytest.approx(T_orc, rel=2e-3)


def test_learn_q_holdout_and_scores(orc):
    """Reading R28 (PAPER.md L89 gives no procedure) as the oracle runs it.  Pinned here is everything but the reading
    itself: the withheld set is a Bernoulli thinning of the SAMPLES by the HOLDOUT stream's uniforms (rebuilt from the
    Philox words, which are pinned against cuRAND); a candidate's score is the root mean square error at the withheld
    samples of the oracle's own full run on the remaining ones at the temperature of the equipartition line; the learned
    q is the argmin."""
    from paper_1811_01604_b200 import synth
    z = synth.grf(48, 40, 6.0, "gaussian", 5)
    m = synth.bernoulli_mask(48, 40, 0.4, 6)
    seed, f = 4242, 0.25
    held = orc.holdout_mask(m, f, seed)
    assert held.dtype == np.uint8 and not held[m == 0].any()
    key = [seed & 0xFFFFFFFF, seed >> 32]
    for n in (0, 1, 2, 3, 4, 777, 48 * 40 - 1):
        u = orc.u01(int(orc.philox4x32_10([n >> 2, 0, 3, 0], key)[n & 3]))
        assert held.flat[n] == (1 if m.flat[n] and u < f else 0)
    frac = held.sum() / m.sum()
    assert abs(frac - f) < 4 * math.sqrt(f * (1 - f) / m.sum())
    assert not np.array_equal(held, orc.holdout_mask(m, f, seed + 1)) and not np.array_equal(held, orc.holdout_mask(m, f, seed, g=1))
    p = orc.Params(seed=seed, equil_cap=150, M=6, sweeps_per_real=3)
    qs = [0.2, 0.5]
    q_hat, scores, Ts = orc.learn_q(z, m, p, qs, f)
    train = (m & (1 - held)).astype(np.uint8)
    import dataclasses
    for q, sc, T in zip(qs, scores, Ts):
        pq = dataclasses.replace(p, q=float(np.float32(q)))
        phi, _, _ = orc.transform(z, train, seed)
        e_s, _ = orc.sample_energy(phi, train, pq.q)
        assert T == orc.default_ladder(48, 40, e_s, (1.0,))[0]
        pred = orc.run(z, train, T, pq)["pred"]
        assert sc == pytest.approx(float(np.sqrt(np.mean((z.astype(np.float64) - pred)[held == 1] ** 2))), rel=1e-12)
    assert q_hat == float(np.float32(qs[int(np.argmin(scores))]))
    assert Ts[0] < Ts[1]               # (1 + e_s) ~ q^2: a smaller q needs a lower temperature for the same data
