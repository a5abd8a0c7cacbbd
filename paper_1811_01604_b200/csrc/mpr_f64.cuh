// mpr_f64.cuh -- the double-precision path (Table 2 against Table 3):
// data, spin state, every site update and the realization sums in double.  Included by mpr_api.cu after
// mpr_device.cuh (Philox, the bitmask helpers and the error flags are shared with the fp32 path; no arithmetic is).
//
// State: v_i = (cos q phi_i, sin q phi_i) as double2, one plane per checkerboard colour (vpos), updated IN PLACE: the
// sites of one colour depend only on the other colour, so a half-sweep is one kernel with one
// thread per PREDICTION site of that colour (the paper's own design, L261-267, gives every lattice site a thread and
// lets those of the sample sites idle; here the prediction sites of each colour are listed once, in row-major order,
// so that every lane of a warp has an update to do).  Measured on cfg4 (profiles/r01h): 62 us per half-sweep, 327 MB
// of DRAM traffic = 5.3 TB/s = 0.82 of the measured HBM peak, fp64 pipe 26 %: this kernel is bound by bytes.  The
// fp32 path's shared-memory tile pass (K sweeps per load) is what would lift it; not built for double yet
// (DESIGN.md section 12).  One grid per context.
#pragma once
#include "mpr_device.cuh"

namespace mpr64 {

using mpr::ERRF_DEGENERATE;
using mpr::ERRF_NONFINITE;
using mpr::ERRF_NO_FREE;
using mpr::ERRF_NO_SAMPLES;
using mpr::MAX_NFIT;
using mpr::PHILOX_ROUNDS;
using mpr::is_fixed;
using mpr::philox4x32_10;

constexpr double TWO_PI_D  = 6.28318530717958647692;   // double nearest 2 pi; state space [0, TWO_PI_D]
constexpr int    E_BLOCKS  = 592;                      // energy partials: fixed, so that the sum order is deterministic
constexpr int    E_THREADS = 256;
constexpr int    MM_BLOCKS = 592;

struct State64 {
    uint32_t t, done, i, realizations;
    uint32_t n_samples, n_free, err_flags, pad;
    uint32_t n_colour[2];     // prediction sites per colour = lengths of the two site lists
    unsigned long long accepted;
    double   a, k, A_last, e_last, T, zmin, zmax, e_query;
    double   e_ring[MAX_NFIT];
};

struct Dev64 {
    State64*  state;
    uint32_t* done_flag;
    double*   partials;       // [max(E_BLOCKS, 4 * MM_BLOCKS)]
    double*   values;         // [N] verbatim copy of the input
    double*   phi;            // [N] Eq. 1 at the sample sites; export buffer at the prediction sites
    uint32_t* bits;           // [words] fixed-site bitmask
    uint32_t* list;           // [n_colour[0]] then [n_colour[1]]: the prediction sites of colour 0, then of colour 1, ascending
    uint32_t* list_counts;    // [2][list_blocks] prediction sites per colour of each block of 32 * LIST_THREADS sites
    uint32_t  list_blocks;
    double2*  vec;            // [2][rows][half] unit vectors, one plane per checkerboard colour (vpos): the CURRENT buffer
    double2*  vec_other;      // the other of the two vector buffers (the tile pass writes it; the host swaps the two)
    int       half;           // ceil(cols / 2): sites of one colour in a row (at most)
    uint32_t  plane;          // rows * half
    double*   acc;            // [N] sum over the realizations of phi
    double*   acc2;           // [N] sum of phi^2 (spread, L212)
    int       rows, cols;
    uint32_t  N, words;
    uint32_t  rk0[PHILOX_ROUNDS], rk1[PHILOX_ROUNDS];
    double    q, inv_q, bc, bs, n_bonds;
    uint32_t  n_f, n_fit, equil_cap;
    double    A_targ, k_a;
};

// Where the vector of site (r, c) lives: the two colours in separate planes, so that a half-sweep reads the OTHER
// colour's plane as a stream and touches its own only at the prediction sites (in one row-major array a 32-byte sector
// holds one site of each colour and every half-sweep streamed both: 346 MB and 70 us per half-sweep of cfg4 against
// 327 MB and 62 us now; DRAM moves 64 bytes at a time, i.e. four sites of a colour, of which one in three is free).
// Neighbours of (r, c) sit in the other plane at o = vpos_other(r, c): up o - half, down o + half,
// left o - 1 + (c & 1), right o + (c & 1).
__device__ __forceinline__ size_t vpos(const Dev64& d, int r, int c)
{
    return (size_t)((r + c) & 1) * d.plane + (size_t)r * d.half + (size_t)(c >> 1);
}
__device__ __forceinline__ size_t vpos_other(const Dev64& d, int r, int c)
{
    return (size_t)(((r + c) & 1) ^ 1) * d.plane + (size_t)r * d.half + (size_t)(c >> 1);
}
__device__ __forceinline__ size_t vpos_n(const Dev64& d, uint32_t n)
{
    const int r = (int)(n / (uint32_t)d.cols);
    return vpos(d, r, (int)(n - (uint32_t)r * (uint32_t)d.cols));
}

// u = (2 (x >> 9) + 1) 2^-24 in (0,1): the same lattice as the fp32 path (R13), exact in double
// built without an integer -> double conversion: f = 1.m in [1, 2) with m = x >> 9 in the top 23 mantissa bits, u = f - (1 - 2^-24)
__device__ __forceinline__ double u01d(uint32_t x)
{
    return __hiloint2double((int)(0x3FF00000u | (x >> 12)), (int)(x >> 9 << 29)) - 0.99999994039535522461;
}

// Eq. 1 in double, the oracle's pinned operation order, clamped to [0, TWO_PI_D]
__device__ __forceinline__ double eq1d(double z, double zmin, double zmax)
{
    const double scale = __ddiv_rn(TWO_PI_D, __dsub_rn(zmax, zmin));
    double p = __dmul_rn(__dsub_rn(z, zmin), scale);
    p = p < 0.0 ? 0.0 : p;
    p = p > TWO_PI_D ? TWO_PI_D : p;
    return p;
}

__device__ __forceinline__ double angle_of_d(double2 v, double inv_q)
{
    double p = atan2(v.y, v.x) * inv_q;
    p = p < 0.0 ? 0.0 : p;
    p = p > TWO_PI_D ? TWO_PI_D : p;
    return p;
}

// ---- a1: min / max over the SAMPLE values (L81), sample count, finiteness --------------------------------------
__global__ void __launch_bounds__(256) k64_minmax(Dev64 d, const double* __restrict__ z, const uint8_t* __restrict__ m)
{
    __shared__ double s_lo[8], s_hi[8];
    __shared__ uint32_t s_cnt[8], s_bad[8];
    double lo = INFINITY, hi = -INFINITY;
    uint32_t cnt = 0, bad = 0;
    for (uint32_t n = blockIdx.x * blockDim.x + threadIdx.x; n < d.N; n += gridDim.x * blockDim.x)
        if (m[n]) {
            const double x = z[n];
            bad |= !isfinite(x);
            lo = fmin(lo, x); hi = fmax(hi, x);
            ++cnt;
        }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        lo = fmin(lo, __shfl_xor_sync(0xFFFFFFFFu, lo, o));
        hi = fmax(hi, __shfl_xor_sync(0xFFFFFFFFu, hi, o));
        cnt += __shfl_xor_sync(0xFFFFFFFFu, cnt, o);
        bad |= __shfl_xor_sync(0xFFFFFFFFu, bad, o);
    }
    const int w = threadIdx.x >> 5;
    if ((threadIdx.x & 31) == 0) { s_lo[w] = lo; s_hi[w] = hi; s_cnt[w] = cnt; s_bad[w] = bad; }
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int k = 1; k < 8; ++k) { lo = fmin(lo, s_lo[k]); hi = fmax(hi, s_hi[k]); cnt += s_cnt[k]; bad |= s_bad[k]; }
        d.partials[4 * blockIdx.x + 0] = lo; d.partials[4 * blockIdx.x + 1] = hi;
        d.partials[4 * blockIdx.x + 2] = (double)cnt; d.partials[4 * blockIdx.x + 3] = (double)bad;
    }
}

__global__ void k64_minmax_finish(Dev64 d, int n_blocks)
{
    State64& s = *d.state;
    double lo = INFINITY, hi = -INFINITY, cnt = 0.0, bad = 0.0;
    for (int b = 0; b < n_blocks; ++b) {
        lo = fmin(lo, d.partials[4 * b]); hi = fmax(hi, d.partials[4 * b + 1]);
        cnt += d.partials[4 * b + 2]; bad += d.partials[4 * b + 3];
    }
    uint32_t err = bad > 0.0 ? ERRF_NONFINITE : 0u;
    s.n_samples = (uint32_t)cnt; s.n_free = d.N - (uint32_t)cnt;
    if (cnt == 0.0) err |= ERRF_NO_SAMPLES;
    else {
        s.zmin = lo; s.zmax = hi;
        if (!(err & ERRF_NONFINITE) && !(hi > lo)) err |= ERRF_DEGENERATE;
    }
    if ((uint32_t)cnt == d.N) err |= ERRF_NO_FREE;
    s.err_flags = err;
    s.t = 0; s.done = 0; s.i = 0; s.realizations = 0; s.accepted = 0ull;
    s.a = 1.0; s.k = -1.0; s.A_last = 0.0; s.e_last = 0.0; s.T = 0.0; s.e_query = 0.0;
    *d.done_flag = 0;
}

// ---- a2: Eq. 1 at the sample sites, fixed-site bitmask, verbatim value copy ------------------------------------
__global__ void __launch_bounds__(256) k64_transform(Dev64 d, const double* __restrict__ values,
                                                     const uint8_t* __restrict__ mask)
{
    const uint32_t n = blockIdx.x * blockDim.x + threadIdx.x;      // < 32 * words
    const State64& s = *d.state;
    bool fixed = false;
    if (n < d.N) {
        const double z = values[n];
        fixed = mask[n] != 0;
        d.values[n] = z;
        d.phi[n] = fixed ? eq1d(z, s.zmin, s.zmax) : 0.0;
    }
    const uint32_t b = __ballot_sync(0xFFFFFFFFu, fixed);
    if ((threadIdx.x & 31) == 0 && (n >> 5) < d.words) d.bits[n >> 5] = b;
}

// The checkerboard split (L261) as two lists of prediction sites.  A thread takes one word of the bitmask (32 sites);
// k64_list_count leaves the per-block counts, k64_list_scan turns them into offsets, k64_list_fill writes the sites.
constexpr int LIST_THREADS = 256;
__device__ __forceinline__ void word_free_masks(const Dev64& d, uint32_t w, uint32_t& f0, uint32_t& f1)
{
    f0 = f1 = 0u;
    if (w >= d.words) return;
    const uint32_t fixed = d.bits[w];
    for (uint32_t b = 0; b < 32u; ++b) {
        const uint32_t n = 32u * w + b;
        if (n >= d.N || ((fixed >> b) & 1u)) continue;
        const uint32_t r = n / (uint32_t)d.cols;
        (((r + (n - r * (uint32_t)d.cols)) & 1u) ? f1 : f0) |= 1u << b;
    }
}
// exclusive scan of (x0, x1) over the block's threads; totals returned through t0, t1
__device__ __forceinline__ void block_scan2(uint32_t& x0, uint32_t& x1, uint32_t& t0, uint32_t& t1)
{
    __shared__ uint32_t w0[LIST_THREADS / 32], w1[LIST_THREADS / 32];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    uint32_t i0 = x0, i1 = x1;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const uint32_t a = __shfl_up_sync(0xFFFFFFFFu, i0, o), b = __shfl_up_sync(0xFFFFFFFFu, i1, o);
        if (lane >= o) { i0 += a; i1 += b; }
    }
    if (lane == 31) { w0[warp] = i0; w1[warp] = i1; }
    __syncthreads();
    uint32_t b0 = 0, b1 = 0, s0 = 0, s1 = 0;
    for (int k = 0; k < LIST_THREADS / 32; ++k) {
        if (k < warp) { b0 += w0[k]; b1 += w1[k]; }
        s0 += w0[k]; s1 += w1[k];
    }
    x0 = b0 + i0 - x0; x1 = b1 + i1 - x1; t0 = s0; t1 = s1;
}
__global__ void __launch_bounds__(LIST_THREADS) k64_list_count(Dev64 d)
{
    uint32_t f0, f1, t0, t1;
    word_free_masks(d, blockIdx.x * LIST_THREADS + threadIdx.x, f0, f1);
    uint32_t c0 = __popc(f0), c1 = __popc(f1);
    block_scan2(c0, c1, t0, t1);
    if (threadIdx.x == 0) { d.list_counts[blockIdx.x] = t0; d.list_counts[d.list_blocks + blockIdx.x] = t1; }
}
__global__ void k64_list_scan(Dev64 d)          // one thread: list_blocks <= 2^31 / 8192 additions
{
    uint32_t run = 0;
    for (int c = 0; c < 2; ++c) {
        const uint32_t start = run;
        for (uint32_t b = 0; b < d.list_blocks; ++b) {
            const uint32_t n = d.list_counts[c * d.list_blocks + b];
            d.list_counts[c * d.list_blocks + b] = run;
            run += n;
        }
        d.state->n_colour[c] = run - start;
    }
}
__global__ void __launch_bounds__(LIST_THREADS) k64_list_fill(Dev64 d)
{
    uint32_t f0, f1, t0, t1;
    const uint32_t w = blockIdx.x * LIST_THREADS + threadIdx.x;
    word_free_masks(d, w, f0, f1);
    uint32_t o0 = __popc(f0), o1 = __popc(f1);
    block_scan2(o0, o1, t0, t1);
    o0 += d.list_counts[blockIdx.x]; o1 += d.list_counts[d.list_blocks + blockIdx.x];
    for (; f0; f0 &= f0 - 1u) d.list[o0++] = 32u * w + (uint32_t)(__ffs(f0) - 1);
    for (; f1; f1 &= f1 - 1u) d.list[o1++] = 32u * w + (uint32_t)(__ffs(f1) - 1);
}

// Alg. 2 step 2.2 (L176): prediction sites ~ U(0, 2 pi) from the INIT stream; unit vectors of every site
__global__ void __launch_bounds__(256) k64_init_state(Dev64 d)
{
    const uint32_t n = blockIdx.x * blockDim.x + threadIdx.x;
    if (n >= d.N) return;
    double p = d.phi[n];
    if (!is_fixed(d.bits, n)) {
        const uint4 x = philox4x32_10(n >> 2, 0u, 0u, 0u, d.rk0, d.rk1);
        const uint32_t w = (n & 3u) == 0 ? x.x : (n & 3u) == 1 ? x.y : (n & 3u) == 2 ? x.z : x.w;
        p = __dmul_rn(TWO_PI_D, u01d(w));
        d.phi[n] = p;
    }
    double sn, cs;
    sincos(__dmul_rn(d.q, p), &sn, &cs);
    d.vec[vpos_n(d, n)] = make_double2(cs, sn);
    d.vec_other[vpos_n(d, n)] = make_double2(cs, sn);        // sample sites are never written again
}

// sin and cos of the half rotation |x| <= q pi / 2 <= pi / 4 by their Maclaurin series, to x^17 and x^16 (truncation
// below 1e-19 and 2e-18 relative at pi / 4): no range reduction and no special cases, a third of the library sincos'
// instructions
// (the coefficients sit in the constant bank: a DFMA takes them as an operand, an immediate double costs two moves)
__constant__ double C_SIN[8] = {2.8114572543455206e-15, -7.6471637318198164e-13, 1.6059043836821613e-10, -2.5052108385441720e-08,
                                2.7557319223985893e-06, -1.9841269841269841e-04, 8.3333333333333332e-03, -1.6666666666666666e-01};
__constant__ double C_COS[8] = {4.7794773323873853e-14, -1.1470745597729725e-11, 2.0876756987868100e-09, -2.7557319223985888e-07,
                                2.4801587301587302e-05, -1.3888888888888889e-03, 4.1666666666666664e-02, -0.5};
__constant__ double C_EXP[12] = {1.6059043836821613e-10, 2.0876756987868100e-09, 2.5052108385441720e-08, 2.7557319223985888e-07,
                                 2.7557319223985893e-06, 2.4801587301587302e-05, 1.9841269841269841e-04, 1.3888888888888889e-03,
                                 8.3333333333333332e-03, 4.1666666666666664e-02, 1.6666666666666666e-01, 0.5};
__constant__ double C_LN2[3] = {1.4426950408889634, 6.93147180369123816490e-01, 1.90821492927058770002e-10};   // log2 e; ln 2 high (low 21 bits zero), low
__device__ __forceinline__ void sincos_small_d(double x, double& s, double& c)
{
    const double x2 = x * x;
    double ps = C_SIN[0], pc = C_COS[0];
#pragma unroll
    for (int k = 1; k < 8; ++k) { ps = fma(x2, ps, C_SIN[k]); pc = fma(x2, pc, C_COS[k]); }       // 1/17! ... -1/3!;  1/16! ... -1/2!
    s = fma(x * x2, ps, x);
    c = fma(x2, pc, 1.0);
}

// exp(x) for x <= 0 as the acceptance test needs it (AP = exp(-dH / T) is compared with r >= 2^-24): x = k ln 2 + r
// with |r| <= ln 2 / 2, Maclaurin series of exp r to r^13 (truncation 4e-18), scaled by 2^k through the exponent
// bits; below 2^-40 the result is returned as 0 (it loses against every r).  No special cases, half the library exp.
__device__ __forceinline__ double exp_nonpos_d(double x)
{
    const double t = x * C_LN2[0];
    const double kd = rint(fmax(t, -40.0));
    double r = fma(-kd, C_LN2[1], x);
    r = fma(-kd, C_LN2[2], r);
    double p = C_EXP[0];                                           // 1/13!
#pragma unroll
    for (int k = 1; k < 12; ++k) p = fma(r, p, C_EXP[k]);         // 1/12! ... 1/2!
    p = fma(r, p, 1.0);
    p = fma(r, p, 1.0);
    const long long bits = (long long)((int)kd + 1023) << 52;     // 2^k, k in [-40, 0]
    return t < -40.0 ? 0.0 : p * __longlong_as_double(bits);
}

// 1 / x by the special-function unit's 20-bit estimate and two Newton steps (a division is 25 instructions and a call)
__device__ __forceinline__ double rcp_d(double x)
{
    double r;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
    r = fma(fma(-x, r, 1.0), r, r);
    r = fma(fma(-x, r, 1.0), r, r);
    return r;
}

// ---- a3: UPDATE of one prediction site (Alg. 1) in vector form, in double ----------------------------
// The same algebra as the fp32 path's update_site, written out again in double.
template <bool QHALF, int ORMODE>
__device__ __forceinline__ double2 update_site_d(double2 v, double2 n_up, double2 n_dn, double2 n_lf, double2 n_rt,
                                                 uint32_t w0, uint32_t w1, double hd_scale, double neg_inv_T,
                                                 double bc, double bs, bool& accepted)
{
    const double hx = (n_up.x + n_dn.x) + (n_lf.x + n_rt.x), hy = (n_up.y + n_dn.y) + (n_lf.y + n_rt.y);
    double px = v.x, py = v.y;
    if (ORMODE == 0) {
        // line 1, over-relaxation: v' = 2 (h.v)/(h.h) h - v keeps h.v (L156, L265; R2); out of [0, 2 pi]: keep the spin
        const double R2 = fma(hx, hx, hy * hy);
        const double dot = fma(px, hx, py * hy);
        const double k = (dot + dot) * rcp_d(R2);                // 0 * inf -> NaN -> kept below (R17)
        const double fx = fma(k, hx, -px), fy = fma(k, hy, -py);
        bool in = fy >= 0.0 && hy >= 0.0;
        if (!QHALF) in = in && (fma(fx, bs, -fy * bc) >= 0.0);
        px = in ? fx : px; py = in ? fy : py;
    } else if (ORMODE == 1) {
        // Eq. 6 as printed (L158), q = 1/2 only
        const double C1 = (n_up.x * n_up.x - n_up.y * n_up.y) + (n_dn.x * n_dn.x - n_dn.y * n_dn.y)
                        + (n_lf.x * n_lf.x - n_lf.y * n_lf.y) + (n_rt.x * n_rt.x - n_rt.y * n_rt.y);
        const double S1 = 2.0 * (n_up.x * n_up.y + n_dn.x * n_dn.y + n_lf.x * n_lf.y + n_rt.x * n_rt.y);
        const double R2 = fma(C1, C1, S1 * S1);
        const double inv = R2 > 0.0 ? rsqrt(R2) : 0.0;
        const double ex = R2 > 0.0 ? C1 * inv : 1.0, ey = S1 * inv;
        double fx = fma(ex, px, ey * py), fy = fma(ey, px, -ex * py);
        if (fy < 0.0) { fx = -fx; fy = -fy; }
        px = fx; py = fy;
    }
    // lines 2-3: rotate by d = q delta = 2 hd, hd = (u - 1/2) q pi / a
    const double hd = (u01d(w0) - 0.5) * hd_scale;
    double sh, ch;
    sincos_small_d(hd, sh, ch);
    const double sh2 = sh + sh;
    const double sd = sh2 * ch, omc = sh2 * sh;                  // sin d, 1 - cos d
    double rx = fma(-sd, py, fma(-omc, px, px));
    double ry = fma(sd, px, fma(-omc, py, py));
    // line 4: dH = -h.(v'' - v') = (1 - cos d)(h.v') + sin d (h x v')
    const double hdotp = fma(hx, px, hy * py);
    const double hcrossp = fma(hx, py, -hy * px);
    double dH = fma(omc, hdotp, sd * hcrossp);
    if (QHALF) {
        if (ry < 0.0) { rx = -rx; ry = -ry; dH = fma(2.0, hdotp, -dH); }     // phi -/+ 2 pi <=> v -> -v (R3)
    } else {
        const bool under = hd < 0.0 && ry < 0.0;
        const bool over = hd > 0.0 && !(ry >= 0.0 && fma(rx, bs, -ry * bc) >= 0.0);
        if (under || over) {
            const double s2 = under ? bs : -bs;
            const double wx = fma(rx, bc, -ry * s2), wy = fma(rx, s2, ry * bc);
            rx = wx; ry = wy;
            dH = hdotp - fma(hx, rx, hy * ry);
        }
    }
    // lines 5-6: AP = min{1, exp(-dH/T)}; accept phi'' if AP > r else keep phi'
    accepted = dH <= 0.0 || exp_nonpos_d(dH * neg_inv_T) > u01d(w1);
    return make_double2(accepted ? rx : px, accepted ? ry : py);
}

// One colour of one sweep (L261-265): one thread per prediction site of the colour (sites[0 .. n_sites)), in place.
template <bool QHALF, int ORMODE>
__global__ void __launch_bounds__(256) k64_halfsweep(Dev64 d, const uint32_t* __restrict__ sites, uint32_t n_sites,
                                                     uint32_t t_off, int count, int check_done)
{
    if (check_done && d.state->done) return;        // the equilibration has stopped (Alg. 2 step 5 loop condition false)
    const uint32_t idx = blockIdx.x * blockDim.x + threadIdx.x;
    bool accepted = false;
    if (idx < n_sites) {
        const uint32_t n = sites[idx];
        const int r = (int)(n / (uint32_t)d.cols), c = (int)(n - (uint32_t)r * (uint32_t)d.cols);
        {
            const State64& s = *d.state;
            const uint32_t t = s.t + t_off;
            const double2 zero = make_double2(0.0, 0.0);                 // open boundary (L109)
            const size_t self = vpos(d, r, c), o = vpos_other(d, r, c);
            const double2 up = r > 0 ? d.vec[o - d.half] : zero, dn = r < d.rows - 1 ? d.vec[o + d.half] : zero;
            const double2 lf = c > 0 ? d.vec[o - 1 + (c & 1)] : zero, rt = c < d.cols - 1 ? d.vec[o + (c & 1)] : zero;
            const uint4 x = philox4x32_10(n, t >> 1, 2u, 0u, d.rk0, d.rk1);
            const uint32_t w0 = (t & 1u) ? x.z : x.x, w1 = (t & 1u) ? x.w : x.y;
            const double hd_scale = d.q * (0.5 * TWO_PI_D) / s.a;
            d.vec[self] = update_site_d<QHALF, ORMODE>(d.vec[self], up, dn, lf, rt, w0, w1, hd_scale, -1.0 / s.T, d.bc, d.bs, accepted);
        }
    }
    if (count) {        // one global atomic per block (one per warp on the same address doubled the kernel's time)
        __shared__ uint32_t s_acc;
        if (threadIdx.x == 0) s_acc = 0;
        __syncthreads();
        const uint32_t n_acc = __popc(__ballot_sync(0xFFFFFFFFu, accepted));
        if ((threadIdx.x & 31) == 0 && n_acc) atomicAdd(&s_acc, n_acc);
        __syncthreads();
        if (threadIdx.x == 0 && s_acc) atomicAdd(&d.state->accepted, (unsigned long long)s_acc);
    }
}

// ---- a5: H = - sum over the colour-1 sites of v . h (every bond joins the two colours; Eq. 2) -------------
__global__ void __launch_bounds__(E_THREADS) k64_energy(Dev64 d)
{
    __shared__ double warp_sum[E_THREADS / 32];
    double sum = 0.0;
    for (int r = blockIdx.x; r < d.rows; r += gridDim.x) {
        double row = 0.0;
        for (int c = ((r + 1) & 1) + 2 * (int)threadIdx.x; c < d.cols; c += 2 * E_THREADS) {
            const double2 v = d.vec[vpos(d, r, c)];
            const size_t o = vpos_other(d, r, c);
            double hx = 0.0, hy = 0.0;
            if (r > 0) { hx += d.vec[o - d.half].x; hy += d.vec[o - d.half].y; }
            if (r < d.rows - 1) { hx += d.vec[o + d.half].x; hy += d.vec[o + d.half].y; }
            if (c > 0) { hx += d.vec[o - 1 + (c & 1)].x; hy += d.vec[o - 1 + (c & 1)].y; }
            if (c < d.cols - 1) { hx += d.vec[o + (c & 1)].x; hy += d.vec[o + (c & 1)].y; }
            row += fma(v.x, hx, v.y * hy);
        }
        sum += row;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) sum += __shfl_xor_sync(0xFFFFFFFFu, sum, o);
    if ((threadIdx.x & 31) == 0) warp_sum[threadIdx.x >> 5] = sum;
    __syncthreads();
    if (threadIdx.x == 0) {
        double s = 0.0;
        for (int w = 0; w < E_THREADS / 32; ++w) s += warp_sum[w];
        d.partials[blockIdx.x] = -s;
    }
}

__device__ __forceinline__ double sum_partials64(const Dev64& d, int n)      // one warp, fixed order
{
    double s = 0.0;
    for (int b = threadIdx.x; b < n; b += 32) s += d.partials[b];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xFFFFFFFFu, s, o);
    return s;
}
__global__ void k64_energy_query(Dev64 d, int n_partials)
{
    const double H = sum_partials64(d, n_partials);
    if (threadIdx.x == 0) d.state->e_query = H / d.n_bonds;
}

// ---- a6: Alg. 2 steps 5.2-5.5 (L195-206) after a counted sweep and its energy -----------------------------------
__global__ void k64_controller(Dev64 d, int n_partials)
{
    State64& s = *d.state;
    if (s.done) return;
    const double H = sum_partials64(d, n_partials);
    if (threadIdx.x != 0) return;
    const uint32_t i = s.i;
    const double A = (double)s.accepted / (double)s.n_free;
    double a = s.a;
    if (A < d.A_targ) a = 1.0 + (double)(i + 1u) / d.k_a;                 // 5.2
    const double e = H / d.n_bonds;                                       // 5.3
    s.e_ring[(i + 1u) % d.n_fit] = e;
    double k = s.k;
    if (i >= d.n_fit && i % d.n_f == 0) {                                 // 5.4: OLS slope of the last n_fit energies (R9)
        const int n = (int)d.n_fit;
        const double tbar = 0.5 * (double)(n - 1);
        double ebar = 0.0;
        for (int j = 0; j < n; ++j) ebar += s.e_ring[(i + 2u - d.n_fit + j) % d.n_fit];
        ebar /= (double)n;
        double num = 0.0, den = 0.0;
        for (int j = 0; j < n; ++j) {
            const double dt = (double)j - tbar;
            num += dt * (s.e_ring[(i + 2u - d.n_fit + j) % d.n_fit] - ebar);
            den += dt * dt;
        }
        k = num / den;
    }
    s.i = i + 1u; s.t += 1u; s.a = a; s.k = k; s.A_last = A; s.e_last = e; s.accepted = 0ull;     // 5.5
    if (!(k < 0.0 && i + 1u < d.equil_cap)) { s.done = 1u; *d.done_flag = 1u; }
}

// ---- a7 / a8 ----------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k64_accumulate(Dev64 d)
{
    const uint32_t n = blockIdx.x * blockDim.x + threadIdx.x;
    if (n >= d.N || is_fixed(d.bits, n)) return;
    const double p = angle_of_d(d.vec[vpos_n(d, n)], d.inv_q);
    d.acc[n] += p; d.acc2[n] += p * p;
}
__global__ void __launch_bounds__(256) k64_predict(Dev64 d, double* __restrict__ out, int what)
{
    const uint32_t n = blockIdx.x * blockDim.x + threadIdx.x;
    if (n >= d.N) return;
    const State64& s = *d.state;
    const double scale = (s.zmax - s.zmin) / TWO_PI_D, M = (double)s.realizations;
    if (what == 0) {            // step 7: mean, back-transformed (L148, L212); sample sites = the input
        out[n] = is_fixed(d.bits, n) ? d.values[n] : s.zmin + (d.acc[n] / M) * scale;
    } else {                    // spread of the realizations: unbiased sample standard deviation
        const double var = fmax((d.acc2[n] - d.acc[n] * d.acc[n] / M) / (M - 1.0), 0.0);
        out[n] = is_fixed(d.bits, n) ? 0.0 : sqrt(var) * scale;
    }
}
__global__ void __launch_bounds__(256) k64_export_angles(Dev64 d)
{
    const uint32_t n = blockIdx.x * blockDim.x + threadIdx.x;
    if (n >= d.N || is_fixed(d.bits, n)) return;
    d.phi[n] = angle_of_d(d.vec[vpos_n(d, n)], d.inv_q);
}
__global__ void __launch_bounds__(256) k64_import_angles(Dev64 d, const double* __restrict__ phi_in)
{
    const uint32_t n = blockIdx.x * blockDim.x + threadIdx.x;
    if (n >= d.N || is_fixed(d.bits, n)) return;
    double p = phi_in[n];
    p = p < 0.0 ? 0.0 : p;
    p = p > TWO_PI_D ? TWO_PI_D : p;
    d.phi[n] = p;
    double sn, cs;
    sincos(__dmul_rn(d.q, p), &sn, &cs);
    d.vec[vpos_n(d, n)] = make_double2(cs, sn);
}
// ---- a3 / a4 in shared memory: K whole sweeps of one tile per launch (temporal blocking, DESIGN.md sections 6, 12) ----
// The fp32 path's tile pass for double vectors.  A tile's frame (core + halo of H sites) is loaded by two TMA tensor loads,
// one per colour plane, into a shared-memory copy with the planes' own layout (element (lr, lc) of colour p at
// S[p][lr * FCH + (lc >> 1)]; out-of-grid elements arrive as zeros: the open boundary, L109); 2K half-sweeps walk the
// prefixes of the tile's entry lists (built by the fp32 path's k_tile_count / k_tile_fill on this grid's bitmask: frame
// offsets lr * FC + lc, core first, then ring by ring), halo sites being recomputed bit for bit because the random
// numbers are keyed by (site, sweep); the core's rows leave by one bulk copy per row and plane into the OTHER vector
// buffer.  Every sweep draws its own Philox block (40 integer instructions against ~250 of double arithmetic per update:
// nothing to save by storing the second pair).  Accepted proposals are not counted here: counted sweeps and the
// equilibration (which needs the energy after every sweep, L199) use k64_halfsweep.
constexpr int T64_THREADS = 512;
__device__ __forceinline__ void tma_load_plane(void* dst, const CUtensorMap* map, int c64, int r, uint64_t* bar)
{
    asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];"
                 ::"r"(mpr::smem_u32(dst)), "l"((uint64_t)map), "r"(c64), "r"(r), "r"(mpr::smem_u32(bar)) : "memory");
}

template <bool QHALF, int ORMODE>
__global__ void __launch_bounds__(T64_THREADS, 2)
k64_tilepass(const __grid_constant__ CUtensorMap map_p0, const __grid_constant__ CUtensorMap map_p1, const Dev64 d,
             const mpr::Dev dt, double2* __restrict__ dst, uint32_t K, uint32_t t_off)
{
    extern __shared__ __align__(128) unsigned char smem64[];
    __shared__ __align__(8) uint64_t s_bar[2];
    __shared__ uint32_t s_cle[2][mpr::MAX_H];
    const int tile = blockIdx.x, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    constexpr int NT = T64_THREADS, NW = T64_THREADS / 32;
    const int H = dt.H, FC = dt.FC, FCH = FC / 2, FR = dt.FR;
    double2* S0 = reinterpret_cast<double2*>(smem64);
    double2* S1 = S0 + FR * FCH;
    uint16_t* E = reinterpret_cast<uint16_t*>(S1 + FR * FCH);
    const mpr::TileGeom tg = mpr::tile_geom(dt, tile);
    const mpr::TileMeta& meta = dt.tile_meta[tile];
    const uint32_t entry_bytes = dt.max_entries * (uint32_t)sizeof(uint16_t);
    if (tid == 0) {
        mpr::mbar_init(&s_bar[0], 1);
        mpr::mbar_expect_tx(&s_bar[0], (uint32_t)(2 * FR * FCH * sizeof(double2)));
        tma_load_plane(S0, &map_p0, tg.c0 - H, tg.r0 - H, &s_bar[0]);      // inner coordinate in 8-byte units: 2 * ((c0 - H) >> 1)
        tma_load_plane(S1, &map_p1, tg.c0 - H, tg.r0 - H, &s_bar[0]);
    } else if (tid == 32) {
        mpr::mbar_init(&s_bar[1], 1);
        mpr::mbar_expect_tx(&s_bar[1], entry_bytes);
        if (entry_bytes) mpr::bulk_load(E, dt.entries + (size_t)tile * dt.tile_entries, entry_bytes, &s_bar[1]);
    }
    if (tid >= 64 && tid < 64 + 2 * mpr::MAX_H) (&s_cle[0][0])[tid - 64] = (&meta.cle[0][0])[tid - 64];
    const State64& st = *d.state;
    const uint32_t t0 = st.t + t_off;
    const double hd_scale = d.q * (0.5 * TWO_PI_D) / st.a, neg_inv_T = -1.0 / st.T;
    __syncthreads();
    mpr::mbar_wait(&s_bar[1], 0);
    mpr::mbar_wait(&s_bar[0], 0);
    const uint32_t base1 = mpr::colour1_base(s_cle[0][mpr::MAX_H - 1]);
#pragma unroll 1
    for (uint32_t j = 0; j < 2u * K; ++j) {
        const uint32_t c = j & 1u, t = t0 + (j >> 1), R = 2u * K - 1u - j;
        const uint32_t n = s_cle[c][R < (uint32_t)mpr::MAX_H ? R : (uint32_t)mpr::MAX_H - 1u];
        const uint16_t* Ec = E + (c ? base1 : 0u);
        double2* own = c ? S1 : S0;
        const double2* oth = c ? S0 : S1;
#pragma unroll 1
        for (uint32_t e = tid; e < n; e += NT) {
            const int off = Ec[e];
            const int lr = (int)(((uint32_t)off * dt.fc_inv) >> 24), lc = off - lr * FC;
            const int o = lr * FCH + (lc >> 1);
            MPR_CHECK(lr >= 1 && lr + 1 < FR && lc >= 1 && lc + 1 < FC && (c ? base1 : 0u) + e < dt.max_entries);
            const double2 up = oth[o - FCH], dn = oth[o + FCH], lf = oth[o - 1 + (lc & 1)], rt = oth[o + (lc & 1)];
            const uint32_t site = (uint32_t)((tg.r0 - H + lr) * d.cols + (tg.c0 - H + lc));
            const uint4 x = philox4x32_10(site, t >> 1, 2u, 0u, d.rk0, d.rk1);
            const uint32_t w0 = (t & 1u) ? x.z : x.x, w1 = (t & 1u) ? x.w : x.y;
            bool accepted;
            own[o] = update_site_d<QHALF, ORMODE>(own[o], up, dn, lf, rt, w0, w1, hd_scale, neg_inv_T, d.bc, d.bs, accepted);
        }
        __syncthreads();
    }
    mpr::fence_proxy_async_smem();
    __syncthreads();
    // the core's rows, one bulk copy per row and plane (both planes take ceil(width / 2) elements: the odd one out is a pad)
    const uint32_t row_bytes = (uint32_t)((tg.TCc + 1) / 2) * (uint32_t)sizeof(double2);
    for (int i = warp + NW * lane; i < 2 * tg.TRc; i += NW * 32) {
        const int p = i & 1, lr = i >> 1;
        const double2* src = (p ? S1 : S0) + (H + lr) * FCH + (H >> 1);
        mpr::bulk_store(dst + (size_t)p * d.plane + (size_t)(tg.r0 + lr) * d.half + (size_t)(tg.c0 >> 1), src, row_bytes);
    }
    mpr::bulk_commit_wait_read();
}

// scalar state edits: what = 0 begin a run at temperature x; 1 set a = x; 2 commit u sweeps (t += u) and v realizations;
// 3 set t = u
__global__ void k64_edit(Dev64 d, int what, double x, uint32_t u, uint32_t v)
{
    State64& s = *d.state;
    if (what == 0) {
        s.t = 0; s.done = 0; s.i = 0; s.realizations = 0; s.accepted = 0ull;
        s.a = 1.0; s.k = -1.0; s.A_last = 0.0; s.e_last = 0.0; s.T = x; *d.done_flag = 0;
    } else if (what == 1) { s.a = x; s.accepted = 0ull; }
    else if (what == 2) { s.t += u; s.realizations += v; }
    else if (what == 3) { s.t = u; }
}

}  // namespace mpr64
