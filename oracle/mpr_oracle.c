/*
 * oracle/mpr_oracle.c -- CPU ORACLE.  TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * A plain, slow, step-by-step restatement of the modified planar rotator (MPR)
 * conditional simulation of arXiv 1811.01604 ("PAPER.md" below), written from
 * the paper, in the paper's order and notation.  It shares no code, header,
 * table or helper with the CUDA path under paper_1811_01604_b200/csrc/ and
 * must never be imported by it.  Only tests/, __graft_entry__.smoke() and the
 * cpu_baseline / --impl reference legs of bench.py may call it.
 *
 * Arithmetic: the spin state is stored in float (as on the GPU; with
 * -DORC_F64 in double, see real_t below); everything
 * inside one site update is done in double from that state and rounded ONCE
 * to the storage type when stored.  The data->angle transform (Eq. 1) alone is done in
 * float with a fixed operation order because the GPU must match it bit for
 * bit.  "2 pi" is the float nearest to 2 pi, TWO_PI = 6.2831854820251465,
 * everywhere (state space [0, TWO_PI]; reading R4).
 *
 * Pins (tests/test_oracle_pins.py): exact energies of hand-built grids,
 * N_GP = 2L(L-1), over-relaxation local-energy conservation and involution,
 * fixed sites bit-identical, Metropolis/Boltzmann chi-square against
 * quadrature, Philox against the cuRAND host generator, uniform lattice,
 * OLS slope closed forms, transform closed forms, unconditional equipartition
 * energy, the sample specific energy of hand-built grids, the unconditional
 * energy of a 2 x 2 grid against 4-D quadrature, and the paper's Table 3
 * validation measures.
 * Parity unpinned (nothing printed in the paper can tell the readings apart):
 * the value of `a` used in equilibrium (R10), the SG filter degree (R9), the
 * defaults of n_f, n_fit, A_targ, k_a (R7), the start and burn-in of the
 * unconditional chains of step 4.2 (R23; their result is pinned).
 *
 * OpenMP (optional, -fopenmp): only over the rows of ONE colour inside a
 * half-sweep and over rows of the energy sum; sites of one colour are
 * independent given the other colour, so the result does not
 * depend on the thread count.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* Storage type of data and spin state.  Default float: the configurations of BASELINE.json and the paper's
 * single-precision program (Table 3).  -DORC_F64 builds the same source with double storage (the paper's
 * double-precision program, Table 2): "2 pi" is then the double nearest 2 pi, Eq. 1 is the
 * same pinned operation order in double, and a site update computes in double from the double state. */
#ifdef ORC_F64
typedef double real_t;
#define ORC_TWO_PI_F 6.28318530717958647692
#else
typedef float real_t;
#define ORC_TWO_PI_F 6.28318530717958647692f
#endif
static const double TWO_PI = (double)ORC_TWO_PI_F;

/* The rows of one colour are swept by OpenMP threads only on grids of at least 4096 sites: a parallel region costs
 * microseconds to milliseconds (on a busy or oversubscribed host), far more than a sweep of the tiny grids the pins use.
 * Scheduling only: the sites of a colour are independent (L261-265), so the result does not depend on the thread
 * count (pinned: test_sweep_independent_of_thread_count). */
#define ORC_PARALLEL(rows, cols) ((long)(rows) * (long)(cols) >= 4096L)
int orc_real_bytes(void) { return (int)sizeof(real_t); }

/* ------------------------------------------------------------------------
 * Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11), the generator the paper
 * names.  counter c[4], key k[2] -> 4 words.
 * ---------------------------------------------------------------------- */
void orc_philox4x32_10(const uint32_t c_in[4], const uint32_t k_in[2], uint32_t out[4])
{
    uint32_t c0 = c_in[0], c1 = c_in[1], c2 = c_in[2], c3 = c_in[3];
    uint32_t k0 = k_in[0], k1 = k_in[1];
    for (int round = 0; round < 10; ++round) {
        uint64_t p0 = (uint64_t)0xD2511F53u * (uint64_t)c0;
        uint64_t p1 = (uint64_t)0xCD9E8D57u * (uint64_t)c2;
        uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
        uint32_t n1 = (uint32_t)p1;
        uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
        uint32_t n3 = (uint32_t)p0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* Uniform in (0,1) from one 32-bit word: (2*(x>>9)+1) * 2^-24.  Exactly
 * representable in float, never 0 or 1, symmetric about 1/2 (reading R13). */
double orc_u01(uint32_t x)
{
    return (double)(2u * (x >> 9) + 1u) * (1.0 / 16777216.0);
}

/* Random-stream layout (reading R13; the paper only says "two numbers per
 * spin per MC step" from Philox4_32_10, L267).  key = (seed_lo, seed_hi).
 *   INIT  stream: counter = (n >> 2, 0, 0, g), word n & 3, n = row*cols+col.
 *   SWEEP stream: counter = (n, t >> 1, 2, g), keyed by the SITE n and the
 *     pair of sweeps (t, t+1): words (x0, x1) give (u, r) at even t, words
 *     (x2, x3) at odd t.  t = global sweep index, increasing from the first
 *     equilibration sweep through all realizations.
 */
static void sweep_uniforms(uint64_t seed, uint32_t g, uint32_t t, uint32_t n,
                           double *u, double *r)
{
    uint32_t ctr[4] = { n, t >> 1, 2u, g };
    uint32_t key[2] = { (uint32_t)seed, (uint32_t)(seed >> 32) };
    uint32_t x[4];
    orc_philox4x32_10(ctr, key, x);
    int slot = (int)(t & 1u);
    *u = orc_u01(x[2 * slot]);
    *r = orc_u01(x[2 * slot + 1]);
}

/* ------------------------------------------------------------------------
 * O1  data -> angle transform, PAPER.md L79-81 (Eq. 1), L181-183 (Alg. 2
 * step 3).  Minimum and maximum over SAMPLE values only.
 * Returns the number of sample sites.
 * ---------------------------------------------------------------------- */
int64_t orc_minmax(const real_t *z, const uint8_t *mask, int64_t n, real_t *zmin, real_t *zmax)
{
    int64_t count = 0;
    real_t lo = INFINITY, hi = -INFINITY;
    for (int64_t i = 0; i < n; ++i) {
        if (!mask[i]) continue;
        if (z[i] < lo) lo = z[i];
        if (z[i] > hi) hi = z[i];
        ++count;
    }
    *zmin = lo; *zmax = hi;
    return count;
}

/* Eq. 1 in float, pinned order (no FMA contraction: build with
 * -ffp-contract=off): scale = TWO_PI_F / (zmax - zmin);
 * phi = (z - zmin) * scale, clamped to [0, TWO_PI_F]. */
real_t orc_eq1(real_t z, real_t zmin, real_t zmax)
{
    volatile real_t range = zmax - zmin;
    volatile real_t scale = ORC_TWO_PI_F / range;
    volatile real_t d = z - zmin;
    real_t phi = d * scale;
    if (phi < 0) phi = 0;
    if (phi > ORC_TWO_PI_F) phi = ORC_TWO_PI_F;
    return phi;
}

/* O1 + O2: sample sites by Eq. 1; prediction sites ~ U(0, 2 pi) from the INIT
 * stream (Alg. 2 step 2.2): phi = TWO_PI_F * u in float (u is
 * exact in float, one rounding). */
void orc_transform(const real_t *z, const uint8_t *mask, int rows, int cols,
                   uint64_t seed, uint32_t g, real_t zmin, real_t zmax, real_t *phi)
{
    uint32_t key[2] = { (uint32_t)seed, (uint32_t)(seed >> 32) };
    for (int64_t n = 0; n < (int64_t)rows * cols; ++n) {
        if (mask[n]) {
            phi[n] = orc_eq1(z[n], zmin, zmax);
        } else {
            uint32_t ctr[4] = { (uint32_t)(n >> 2), 0u, 0u, g };
            uint32_t x[4];
            orc_philox4x32_10(ctr, key, x);
            real_t u = (real_t)orc_u01(x[n & 3]);
            volatile real_t p = ORC_TWO_PI_F * u;
            phi[n] = p;
        }
    }
}

/* ------------------------------------------------------------------------
 * Local quantities of one site given its neighbours' field
 *   C = sum_j cos(q phi_j),  S = sum_j sin(q phi_j)
 * sum_j cos[q(phi - phi_j)] = C cos(q phi) + S sin(q phi); J = 1 (L95).
 * ---------------------------------------------------------------------- */
double orc_local_energy(double phi, double C, double S, double q)
{
    return -(C * cos(q * phi) + S * sin(q * phi));
}

/* Over-relaxation step R, PAPER.md L156-160 (Eq. 6), L119 (Alg. 1 line 1).
 * mode 0 (default, reading R2): exact reflection for the coupling
 *   cos[q(phi_i - phi_j)]: phi' = (2/q) atan2(S, C) - phi, which keeps
 *   C cos(q phi) + S sin(q phi) unchanged; if phi' falls outside [0, 2 pi] the
 *   spin is kept (the only other energy-equal angles are phi' +- 4 pi k / (2q)).
 * mode 1: Eq. 6 as printed: phi' = [2 atan2(sum sin phi_j, sum cos phi_j)
 *   - phi] mod 2 pi; (C1, S1) are those q-less sums.
 * mode 2: no over-relaxation.
 * *kept = 1 when the reflection was rejected (mode 0) / not applied. */
double orc_or_reflect(double phi, double C, double S, double C1, double S1,
                      double q, int mode, int *kept, double *phi_raw)
{
    double p;
    *kept = 0;
    if (mode == 0) {
        double Theta = atan2(S, C);
        p = (2.0 / q) * Theta - phi;
        if (phi_raw) *phi_raw = p;
        if (p < 0.0 || p > TWO_PI) { p = phi; *kept = 1; }
    } else if (mode == 1) {
        p = 2.0 * atan2(S1, C1) - phi;
        if (phi_raw) *phi_raw = p;
        p = fmod(p, TWO_PI);
        if (p < 0.0) p += TWO_PI;
    } else {
        p = phi;
        if (phi_raw) *phi_raw = p;
        *kept = 1;
    }
    return p;
}

/* ------------------------------------------------------------------------
 * O3  UPDATE, PAPER.md L113-146 (Alg. 1) vectorised by the checkerboard
 * decomposition (L261-265): colour 0 = (row+col) even (contains the
 * upper-left node, Fig. 1) first, then colour 1.  One call = one sweep at
 * global sweep index t.  Returns the number of accepted Metropolis proposals.
 *
 * Optional per-site diagnostics (row-major double arrays, may be NULL):
 *   d_margin[n] = |AP - r|                       (Metropolis decision margin)
 *   d_edge[n]   = min distance of the raw reflected angle and of the
 *                 unwrapped proposal to the interval ends 0 and 2 pi
 *   d_R[n]      = sqrt(C^2 + S^2)                 (conditioning of atan2)
 * ---------------------------------------------------------------------- */
static double dist_to_ends(double x)
{
    double a = fabs(x), b = fabs(x - TWO_PI);
    return a < b ? a : b;
}

uint64_t orc_sweep(real_t *phi, const uint8_t *mask, int rows, int cols,
                   double q, double T, double a, uint64_t seed, uint32_t g,
                   uint32_t t, int or_mode,
                   double *d_margin, double *d_edge, double *d_R)
{
    uint64_t accepted_total = 0;
    for (int colour = 0; colour < 2; ++colour) {
        uint64_t accepted = 0;
#ifdef _OPENMP
#pragma omp parallel for schedule(static) reduction(+:accepted) if(ORC_PARALLEL(rows, cols))
#endif
        for (int r = 0; r < rows; ++r) {
            for (int c = (r + colour) & 1; c < cols; c += 2) {
                int64_t n = (int64_t)r * cols + c;
                if (mask[n]) continue;               /* sample sites stay fixed (L148) */
                /* neighbours' field, open boundaries (L109) */
                double C = 0.0, S = 0.0, C1 = 0.0, S1 = 0.0;
                if (r > 0)        { double pj = phi[n - cols]; C += cos(q * pj); S += sin(q * pj); C1 += cos(pj); S1 += sin(pj); }
                if (r < rows - 1) { double pj = phi[n + cols]; C += cos(q * pj); S += sin(q * pj); C1 += cos(pj); S1 += sin(pj); }
                if (c > 0)        { double pj = phi[n - 1];    C += cos(q * pj); S += sin(q * pj); C1 += cos(pj); S1 += sin(pj); }
                if (c < cols - 1) { double pj = phi[n + 1];    C += cos(q * pj); S += sin(q * pj); C1 += cos(pj); S1 += sin(pj); }
                double p_old = (double)phi[n];
                /* Alg. 1 line 1: over-relaxation */
                int kept; double p_raw;
                double p1 = orc_or_reflect(p_old, C, S, C1, S1, q, or_mode, &kept, &p_raw);
                /* line 2: u ~ U(0,1);  line 6: r ~ U(0,1) */
                double u, rr;
                sweep_uniforms(seed, g, t, (uint32_t)n, &u, &rr);
                /* line 3: phi'' = phi' + 2 pi (u - 0.5)/a (mod 2 pi) */
                double p2_raw = p1 + TWO_PI * (u - 0.5) / a;
                double p2 = p2_raw;
                if (p2 < 0.0) p2 += TWO_PI;
                else if (p2 >= TWO_PI) p2 -= TWO_PI;
                /* line 4: Delta H = H(phi'') - H(phi') (local) */
                double dH = orc_local_energy(p2, C, S, q) - orc_local_energy(p1, C, S, q);
                /* line 5: AP = min{1, exp(-Delta H / T)} */
                double AP = exp(-dH / T);
                if (AP > 1.0) AP = 1.0;
                /* lines 6-6.2 */
                double p_new;
                if (AP > rr) { p_new = p2; ++accepted; } else { p_new = p1; }
                phi[n] = (real_t)p_new;
                if (d_margin) d_margin[n] = fabs(AP - rr);
                if (d_edge) {
                    double e1 = (or_mode == 0) ? dist_to_ends(p_raw) : 1e30;
                    double e2 = dist_to_ends(p2_raw);
                    d_edge[n] = e1 < e2 ? e1 : e2;
                }
                if (d_R) d_R[n] = sqrt(C * C + S * S);
            }
        }
        accepted_total += accepted;
    }
    return accepted_total;
}

/* ------------------------------------------------------------------------
 * O4  energy, PAPER.md L87 (Eq. 2), J = 1, all in-grid bonds, open
 * boundaries.  N_GP = rows(cols-1) + cols(rows-1) = 2L(L-1) (L109).
 * ---------------------------------------------------------------------- */
int64_t orc_n_bonds(int rows, int cols)
{
    return (int64_t)rows * (cols - 1) + (int64_t)cols * (rows - 1);
}

double orc_energy(const real_t *phi, int rows, int cols, double q)
{
    double *row_sum = (double *)malloc(sizeof(double) * (size_t)rows);
#ifdef _OPENMP
#pragma omp parallel for schedule(static) if(ORC_PARALLEL(rows, cols))
#endif
    for (int r = 0; r < rows; ++r) {
        double h = 0.0;
        for (int c = 0; c < cols; ++c) {
            int64_t n = (int64_t)r * cols + c;
            double p = (double)phi[n];
            if (c < cols - 1) h -= cos(q * (p - (double)phi[n + 1]));
            if (r < rows - 1) h -= cos(q * (p - (double)phi[n + cols]));
        }
        row_sum[r] = h;
    }
    double H = 0.0;
    for (int r = 0; r < rows; ++r) H += row_sum[r];
    free(row_sum);
    return H;
}

/* ------------------------------------------------------------------------
 * Alg. 2 step 4.1, PAPER.md L101-104 (Eq. 4): sample specific energy
 *   e_s = -(1/N_SP) sum over nearest-neighbour pairs of SAMPLE sites of
 *         cos q(phi_i - phi_j),
 * every unordered pair once, N_SP their number (reading R1).
 * Returns e_s (0 when there is no such pair) and N_SP through n_pairs.
 * ---------------------------------------------------------------------- */
double orc_sample_energy(const real_t *phi, const uint8_t *mask, int rows, int cols,
                         double q, int64_t *n_pairs)
{
    double sum = 0.0;
    int64_t n_sp = 0;
    for (int r = 0; r < rows; ++r)
        for (int c = 0; c < cols; ++c) {
            int64_t n = (int64_t)r * cols + c;
            if (!mask[n]) continue;
            double p = (double)phi[n];
            if (c < cols - 1 && mask[n + 1]) { sum += cos(q * (p - (double)phi[n + 1])); ++n_sp; }
            if (r < rows - 1 && mask[n + cols]) { sum += cos(q * (p - (double)phi[n + cols])); ++n_sp; }
        }
    *n_pairs = n_sp;
    return n_sp ? -sum / (double)n_sp : 0.0;
}

/* ------------------------------------------------------------------------
 * Slope of the energy evolution: Savitzky-Golay
 * first-derivative filter of degree 1 over the window = ordinary least
 * squares slope through (0, e0) ... (n-1, e_{n-1})  (reading R9).
 * ---------------------------------------------------------------------- */
double orc_sg_slope(const double *e, int n)
{
    double tbar = 0.5 * (double)(n - 1), ebar = 0.0;
    for (int j = 0; j < n; ++j) ebar += e[j];
    ebar /= (double)n;
    double num = 0.0, den = 0.0;
    for (int j = 0; j < n; ++j) {
        num += ((double)j - tbar) * (e[j] - ebar);
        den += ((double)j - tbar) * ((double)j - tbar);
    }
    return num / den;
}

static int64_t count_free(const uint8_t *mask, int64_t n)
{
    int64_t P = 0;
    for (int64_t i = 0; i < n; ++i) if (!mask[i]) ++P;
    return P;
}

/* ------------------------------------------------------------------------
 * O5  non-equilibrium relaxation, PAPER.md L192-206 (Alg. 2 step 5).
 *   i = 0, a = 1, k = -1
 *   while k < 0 and i < cap:
 *     5.1 UPDATE at a(i)
 *     5.2 if A < A_targ: a(i+1) = 1 + (i+1)/k_a         (A = accepted / P)
 *     5.3 e(i+1) = H / N_GP
 *     5.4 if i >= n_fit and i mod n_f == 0: k = slope of the last n_fit e's
 *     5.5 i = i + 1
 * History (length >= cap+1 each, may be NULL): e_hist[i+1], A_hist[i+1],
 * a_hist[i+1] = a after step 5.2.  *t_io is the global sweep index.
 * Returns i = number of sweeps done.
 * ---------------------------------------------------------------------- */
int orc_equilibrate(real_t *phi, const uint8_t *mask, int rows, int cols,
                    double q, double T, uint64_t seed, uint32_t g, int or_mode,
                    int cap, int n_f, int n_fit, double A_targ, double k_a,
                    uint32_t *t_io, double *a_out, double *k_out,
                    double *e_hist, double *A_hist, double *a_hist)
{
    int64_t P = count_free(mask, (int64_t)rows * cols);
    int64_t NGP = orc_n_bonds(rows, cols);
    double *e = (double *)malloc(sizeof(double) * (size_t)(cap + 2));
    int i = 0;
    double a = 1.0, k = -1.0;
    uint32_t t = *t_io;
    e[0] = orc_energy(phi, rows, cols, q) / (double)NGP;
    if (e_hist) { e_hist[0] = e[0]; A_hist[0] = 0.0; a_hist[0] = a; }
    while (k < 0.0 && i < cap) {
        uint64_t acc = orc_sweep(phi, mask, rows, cols, q, T, a, seed, g, t, or_mode, NULL, NULL, NULL);
        ++t;
        double A = (double)acc / (double)P;
        if (A < A_targ) a = 1.0 + (double)(i + 1) / k_a;
        e[i + 1] = orc_energy(phi, rows, cols, q) / (double)NGP;
        if (i >= n_fit && i % n_f == 0) k = orc_sg_slope(&e[i + 2 - n_fit], n_fit);
        if (e_hist) { e_hist[i + 1] = e[i + 1]; A_hist[i + 1] = A; a_hist[i + 1] = a; }
        ++i;
    }
    free(e);
    *t_io = t; *a_out = a; *k_out = k;
    return i;
}

/* ------------------------------------------------------------------------
 * O6  equilibrium realizations, PAPER.md L207-211 (Alg. 2 step 6): M times
 * {s sweeps at a_eq; add the state at the prediction sites to acc}.  The
 * paper has s = 1 (L210); BASELINE.json's configurations set s = 100 (R11).
 * acc: double [rows*cols], caller-zeroed; only prediction sites are touched.
 * ---------------------------------------------------------------------- */
/* acc2 (may be NULL): sum over the realizations of phi^2, for the spread of the realizations
 * ("Statistics of M realizations"). */
void orc_simulate2(real_t *phi, const uint8_t *mask, int rows, int cols,
                   double q, double T, double a_eq, uint64_t seed, uint32_t g,
                   int or_mode, int M, int s, uint32_t *t_io, double *acc, double *acc2)
{
    uint32_t t = *t_io;
    int64_t N = (int64_t)rows * cols;
    for (int j = 0; j < M; ++j) {
        for (int w = 0; w < s; ++w) {
            orc_sweep(phi, mask, rows, cols, q, T, a_eq, seed, g, t, or_mode, NULL, NULL, NULL);
            ++t;
        }
        for (int64_t n = 0; n < N; ++n)
            if (!mask[n]) {
                acc[n] += (double)phi[n];
                if (acc2) acc2[n] += (double)phi[n] * (double)phi[n];
            }
    }
    *t_io = t;
}

void orc_simulate(real_t *phi, const uint8_t *mask, int rows, int cols,
                  double q, double T, double a_eq, uint64_t seed, uint32_t g,
                  int or_mode, int M, int s, uint32_t *t_io, double *acc)
{
    orc_simulate2(phi, mask, rows, cols, q, T, a_eq, seed, g, or_mode, M, s, t_io, acc, NULL);
}

/* ------------------------------------------------------------------------
 * O7  prediction, PAPER.md L148 ("mean of the resulting conditional
 * distribution"), L210-212 (Alg. 2 steps 6.3, 7).  The back-transform is
 * linear, so the mean of the back-transformed realizations is the
 * back-transform of the mean angle: z = zmin + mean(phi) (zmax-zmin)/(2 pi).
 * Sample sites return their input value unchanged.
 * ---------------------------------------------------------------------- */
void orc_predict(const double *acc, int M, const real_t *z, const uint8_t *mask,
                 int64_t n_sites, real_t zmin, real_t zmax, real_t *out)
{
    for (int64_t n = 0; n < n_sites; ++n) {
        if (mask[n]) { out[n] = z[n]; continue; }
        double mean_phi = acc[n] / (double)M;
        out[n] = (real_t)((double)zmin + mean_phi * ((double)zmax - (double)zmin) / TWO_PI);
    }
}

/* ------------------------------------------------------------------------
 * Spread of the M realizations at every prediction site (Alg. 2 step 7 "Statistics of M
 * realizations"; L148: the realizations sample the conditional distribution): the unbiased sample standard
 * deviation of the back-transformed values, s_z = sqrt((sum phi^2 - (sum phi)^2 / M) / (M - 1)) (zmax - zmin) / (2 pi),
 * M >= 2; 0 at sample sites (their value is data).
 * ---------------------------------------------------------------------- */
void orc_predict_std(const double *acc, const double *acc2, int M, const uint8_t *mask,
                     int64_t n_sites, real_t zmin, real_t zmax, real_t *out)
{
    for (int64_t n = 0; n < n_sites; ++n) {
        if (mask[n]) { out[n] = 0; continue; }
        double var = (acc2[n] - acc[n] * acc[n] / (double)M) / (double)(M - 1);
        if (var < 0.0) var = 0.0;
        out[n] = (real_t)(sqrt(var) * ((double)zmax - (double)zmin) / TWO_PI);
    }
}

/* ------------------------------------------------------------------------
 * Quantiles of the conditional distribution at the prediction sites from the first two moments of the M
 * realizations ("Statistics of M realizations"; SURVEY 8(f) NEXT-2 "quantiles from sum phi^2";
 * DESIGN.md reading R26): the Gaussian quantile z_p = mean_z + Phi^-1(p) s_z, clamped to the data range
 * [zmin, zmax] that the state space [0, 2 pi] maps to.  Phi^-1 by bisection on Phi(x) = erfc(-x / sqrt 2) / 2.
 * Sample sites return their input value.  0 < p < 1, M >= 2.
 * ---------------------------------------------------------------------- */
double orc_inv_norm_cdf(double p)
{
    double lo = -40.0, hi = 40.0;
    for (int it = 0; it < 200; ++it) {
        double mid = 0.5 * (lo + hi);
        if (0.5 * erfc(-mid / sqrt(2.0)) < p) lo = mid; else hi = mid;
    }
    return 0.5 * (lo + hi);
}

void orc_predict_quantile(const double *acc, const double *acc2, int M, double p, const real_t *z,
                          const uint8_t *mask, int64_t n_sites, real_t zmin, real_t zmax, real_t *out)
{
    const double xp = orc_inv_norm_cdf(p);
    const double scale = ((double)zmax - (double)zmin) / TWO_PI;
    for (int64_t n = 0; n < n_sites; ++n) {
        if (mask[n]) { out[n] = z[n]; continue; }
        double var = (acc2[n] - acc[n] * acc[n] / (double)M) / (double)(M - 1);
        if (var < 0.0) var = 0.0;
        double zq = (double)zmin + (acc[n] / (double)M) * scale + xp * sqrt(var) * scale;
        if (zq < (double)zmin) zq = (double)zmin;
        if (zq > (double)zmax) zq = (double)zmax;
        out[n] = (real_t)zq;
    }
}

int orc_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void orc_set_num_threads(int n)
{
#ifdef _OPENMP
    omp_set_num_threads(n);
#else
    (void)n;
#endif
}
