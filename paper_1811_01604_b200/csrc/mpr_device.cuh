// mpr_device.cuh -- device-side data layout and kernels of the MPR hot path
// (sm_100a).  See DESIGN.md "Data layout in HBM" and "Kernels".
//
// State representation.  The spin of site i is kept as the unit vector
//   v_i = (cos q phi_i, sin q phi_i)
// because every quantity of Alg. 1 is a function of
// q phi: the neighbours' field (C, S) = sum_j v_j, the local energy
// -(C cos q phi + S sin q phi) = -h . v (Eq. 2), the over-relaxation
// reflection about h (Eq. 6 generalised to the coupling cos q(phi_i - phi_j),
// DESIGN.md R2) and the Metropolis rotation by q delta (L121).  phi is
// recovered as atan2(v.y, v.x) / q only where the method needs the angle
// itself (realization accumulation, export).
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace mpr {

constexpr float    TWO_PI_F      = 6.28318530717958647692f;  // float nearest 2 pi; state space [0, TWO_PI_F]
constexpr int      MAX_NFIT      = 256;
constexpr uint32_t LIST_SENTINEL = 0xFFFFFFFFu;
constexpr int      TILE_THREADS  = 512;
constexpr int      MAX_H         = 16;                       // largest halo: up to 8 sweeps per tile pass
constexpr int      ENERGY_BLOCKS = 592;                      // 4 x 148 SMs; fixed so the sum order is deterministic
constexpr int      ENERGY_THREADS = 256;

enum : uint32_t { ERRF_NO_SAMPLES = 1u, ERRF_NO_FREE = 2u, ERRF_DEGENERATE = 4u, ERRF_NONFINITE = 8u };
// k_tilepass flags
enum : uint32_t { PASS_COUNT = 1u, PASS_ENERGY = 2u, PASS_ACCUMULATE = 4u, PASS_CHECK_DONE = 8u };

// One per grid, in the workspace.
struct GridState {
    // --- read by every tile pass ---
    uint32_t t;                  // global sweep index (Philox counter word 1 is t >> 1)
    uint32_t done;               // equilibration stopped (Alg. 2 step 5 loop condition false)
    uint32_t cur;                // which of the two vector buffers holds the current state
    float    hd_scale;           // q * pi / a: half of the rotation q*delta per unit (u - 1/2)
    float    neg_log2e_over_T;   // AP = 2^(dH * this)
    uint32_t n_free[2];          // prediction sites per colour
    uint32_t max_tile_entries;   // largest free-site count of one tile frame
    // --- reductions ---
    unsigned long long accepted; // accepted Metropolis proposals since last reset
    uint32_t zmin_enc, zmax_enc; // order-preserving encodings for atomicMin/Max
    uint32_t n_samples;
    uint32_t err_flags;
    // --- Alg. 2 scalars ---
    uint32_t i;                  // equilibration sweeps done
    uint32_t realizations;
    double   a, k, A_last, e_last, T;
    float    zmin, zmax;
    double   e_query;            // result slot of mpr_energy
    double   e_ring[MAX_NFIT];   // e(i) at slot i % n_fit
};

// Free sites of one tile frame (core + halo), see k_tile_fill.
struct TileMeta {
    uint32_t base;                    // offset of the tile's entries in Dev::entries (per grid)
    uint32_t cge[2][MAX_H + 1];       // cge[c][k] = entries of colour c with ring >= k (ring = distance outside the core)
};

// Device view of one context (passed by value to kernels).
struct Dev {
    GridState* states;
    uint32_t*  done_flags;     // [batch] copy of GridState::done for cheap host polling
    double*    e_partials;     // [batch][n_partials]
    float*     values;         // [batch][N] verbatim copy of the input values
    float*     phi;            // [batch][N] angle view: Eq. 1 at sample sites (never rewritten), export buffer at free sites
    uint32_t*  bits;           // [batch][words] fixed-site bitmask
    float2*    vec;            // [2 buffers][batch][2 colours][VS] colour-split padded unit vectors; pad = (0,0)
    uint32_t*  lists;          // [batch][2][LC] padded index | parity<<31 of the free sites, row-major order
    float*     acc;            // [batch][2][VS] sum over realizations of phi at free sites (same index as vec)
    uint32_t*  rowstart;       // [batch][2][rows+1] ordinal of the first free site of each row
    TileMeta*  tile_meta;      // [batch][ntiles]
    uint32_t*  entries;        // [batch][entry_stride] tile frames' free sites: off | local row << 16
    int        batch, rows, cols;
    uint32_t   N, words, W, Wp, VS, LC;
    size_t     VB;             // float2 elements per vector buffer = batch * 2 * VS
    size_t     entry_stride;
    uint32_t   n_partials;
    // tiling
    int        TR, TC, H, FR, FC, ntx, nty, ntiles;
    uint32_t   max_entries;    // smem capacity for entries (even)
    int        use_spare;      // keep the odd sweep's random words in shared memory
    uint32_t   key0, key1;     // Philox key = (seed lo, seed hi)
    float      q, inv_q;
    float      bc, bs;         // (cos 2 pi q, sin 2 pi q): upper end of the q*phi range
    // Alg. 2 controller constants
    uint32_t   n_f, n_fit, equil_cap;
    double     A_targ, k_a, n_bonds;
};

__device__ __forceinline__ float2* cur_vec(const Dev& d, int g, uint32_t which)
{
    return d.vec + (size_t)which * d.VB + (size_t)g * 2 * d.VS;
}

// ---------------------------------------------------------------------------
// Philox4x32-10 (Salmon et al., SC'11), the generator PAPER.md L267 names.
// ---------------------------------------------------------------------------
__device__ __forceinline__ uint4 philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                               uint32_t k0, uint32_t k1)
{
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint32_t hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
        const uint32_t hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
        const uint32_t n0 = hi1 ^ c1 ^ k0;
        const uint32_t n2 = hi0 ^ c3 ^ k1;
        c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
    }
    return make_uint4(c0, c1, c2, c3);
}

// Uniform u = (2 (x >> 9) + 1) 2^-24 in (0,1) (R13), built without
// an integer->float conversion: f = 1.m in [1,2) with m = x >> 9, so
// u = (f - 1) + 2^-24 and u - 1/2 = (f - 1.5) + 2^-24, every step exact.
__device__ __forceinline__ float u01(uint32_t x)
{
    const float f = __uint_as_float(0x3F800000u | (x >> 9));
    return __fadd_rn(__fadd_rn(f, -1.0f), 5.9604644775390625e-08f);
}
__device__ __forceinline__ float u01_centered(uint32_t x)
{
    const float f = __uint_as_float(0x3F800000u | (x >> 9));
    return __fadd_rn(__fadd_rn(f, -1.5f), 5.9604644775390625e-08f);
}

__device__ __forceinline__ float ex2_approx(float x)
{
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// sin and cos of a half-rotation |x| <= q pi / 2 <= pi/4 by their Maclaurin
// series (truncation < 2e-9 relative at pi/4).
__device__ __forceinline__ void sincos_small(float x, float& s, float& c)
{
    const float x2 = x * x;
    float ps = fmaf(x2, 2.75573192e-6f, -1.98412698e-4f);
    ps = fmaf(x2, ps, 8.33333333e-3f);
    ps = fmaf(x2, ps, -1.66666667e-1f);
    s = fmaf(x * x2, ps, x);
    float pc = fmaf(x2, -2.75573192e-7f, 2.48015873e-5f);
    pc = fmaf(x2, pc, -1.38888889e-3f);
    pc = fmaf(x2, pc, 4.16666667e-2f);
    pc = fmaf(x2, pc, -0.5f);
    c = fmaf(x2, pc, 1.0f);
}

__device__ __forceinline__ uint32_t enc_ordered(float f)
{
    const uint32_t b = __float_as_uint(f);
    return (b & 0x80000000u) ? ~b : (b | 0x80000000u);
}
__device__ __forceinline__ float dec_ordered(uint32_t e)
{
    return __uint_as_float((e & 0x80000000u) ? (e & 0x7FFFFFFFu) : ~e);
}

// Eq. 1 in float with a pinned operation order, clamped to
// [0, TWO_PI_F] (R4).
__device__ __forceinline__ float eq1(float z, float zmin, float zmax)
{
    const float scale = __fdiv_rn(TWO_PI_F, __fsub_rn(zmax, zmin));
    float p = __fmul_rn(__fsub_rn(z, zmin), scale);
    p = p < 0.0f ? 0.0f : p;
    p = p > TWO_PI_F ? TWO_PI_F : p;
    return p;
}

__device__ __forceinline__ float angle_of(float2 v, float inv_q)
{
    float p = atan2f(v.y, v.x) * inv_q;
    p = p < 0.0f ? 0.0f : p;
    p = p > TWO_PI_F ? TWO_PI_F : p;
    return p;
}

// padded colour-split index of site (r, col): colour = (r+col)&1, slot (r+1)*Wp + (col>>1) + 1
__device__ __forceinline__ uint32_t padded_index(uint32_t r, uint32_t col, uint32_t Wp)
{
    return (r + 1u) * Wp + (col >> 1) + 1u;
}

// ---------------------------------------------------------------------------
// a1  min / max over the SAMPLE values, sample count, finiteness
// ---------------------------------------------------------------------------
__global__ void k_state_reset(Dev d)
{
    const int g = blockIdx.x * blockDim.x + threadIdx.x;
    if (g >= d.batch) return;
    GridState& s = d.states[g];
    s.t = 0; s.done = 0; s.cur = 0; s.hd_scale = 0.f; s.neg_log2e_over_T = 0.f;
    s.n_free[0] = s.n_free[1] = 0; s.max_tile_entries = 0;
    s.accepted = 0ull;
    s.zmin_enc = 0xFFFFFFFFu; s.zmax_enc = 0u;
    s.n_samples = 0; s.err_flags = 0; s.i = 0; s.realizations = 0;
    s.a = 1.0; s.k = -1.0; s.A_last = 0.0; s.e_last = 0.0; s.T = 0.0;
    s.zmin = 0.f; s.zmax = 0.f; s.e_query = 0.0;
    d.done_flags[g] = 0;
}

__global__ void __launch_bounds__(256) k_minmax(Dev d, const float* __restrict__ values,
                                                const uint8_t* __restrict__ mask)
{
    const int g = blockIdx.y;
    const float*   z = values + (size_t)g * d.N;
    const uint8_t* m = mask + (size_t)g * d.N;
    float lo = INFINITY, hi = -INFINITY;
    uint32_t cnt = 0, bad = 0;
    for (uint32_t n = blockIdx.x * blockDim.x + threadIdx.x; n < d.N; n += gridDim.x * blockDim.x) {
        if (m[n]) {
            const float x = z[n];
            bad |= !isfinite(x);
            lo = fminf(lo, x); hi = fmaxf(hi, x);
            ++cnt;
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        lo = fminf(lo, __shfl_xor_sync(0xFFFFFFFFu, lo, o));
        hi = fmaxf(hi, __shfl_xor_sync(0xFFFFFFFFu, hi, o));
        cnt += __shfl_xor_sync(0xFFFFFFFFu, cnt, o);
        bad |= __shfl_xor_sync(0xFFFFFFFFu, bad, o);
    }
    if ((threadIdx.x & 31) == 0 && cnt) {
        GridState& s = d.states[g];
        atomicMin(&s.zmin_enc, enc_ordered(lo));
        atomicMax(&s.zmax_enc, enc_ordered(hi));
        atomicAdd(&s.n_samples, cnt);
        if (bad) atomicOr(&s.err_flags, ERRF_NONFINITE);
    }
}

__global__ void k_minmax_finish(Dev d)
{
    const int g = blockIdx.x * blockDim.x + threadIdx.x;
    if (g >= d.batch) return;
    GridState& s = d.states[g];
    uint32_t err = s.err_flags;
    if (s.n_samples == 0) err |= ERRF_NO_SAMPLES;
    else {
        s.zmin = dec_ordered(s.zmin_enc);
        s.zmax = dec_ordered(s.zmax_enc);
        if (!(err & ERRF_NONFINITE) && !(s.zmax > s.zmin)) err |= ERRF_DEGENERATE;
    }
    if (s.n_samples == d.N) err |= ERRF_NO_FREE;
    s.err_flags = err;
}

// ---------------------------------------------------------------------------
// a2  Eq. 1 at the sample sites, fixed-site bitmask, verbatim value copy
// ---------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_transform(Dev d, const float* __restrict__ values,
                                                   const uint8_t* __restrict__ mask)
{
    const int g = blockIdx.y;
    const uint32_t n = blockIdx.x * blockDim.x + threadIdx.x;   // < 32 * words (grid sized so)
    const GridState& s = d.states[g];
    const bool in = n < d.N;
    bool fixed = false;
    if (in) {
        const size_t o = (size_t)g * d.N + n;
        const float z = values[o];
        fixed = mask[o] != 0;
        d.values[o] = z;
        d.phi[o] = fixed ? eq1(z, s.zmin, s.zmax) : 0.0f;
    }
    const uint32_t b = __ballot_sync(0xFFFFFFFFu, fixed);
    if ((threadIdx.x & 31) == 0 && (n >> 5) < d.words) d.bits[(size_t)g * d.words + (n >> 5)] = b;
}

// ---------------------------------------------------------------------------
// a2  checkerboard-split lists of the prediction sites: for
// each colour, the free sites in row-major order; the position in the list is
// the site's ordinal o, which keys its random numbers (R13).
// ---------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_rowcount(Dev d)
{
    const int g = blockIdx.y;
    const uint32_t r = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const uint32_t lane = threadIdx.x & 31;
    if (r >= (uint32_t)d.rows) return;
    const uint32_t* bits = d.bits + (size_t)g * d.words;
    uint32_t cnt0 = 0, cnt1 = 0;
    for (uint32_t col = lane; col < (uint32_t)d.cols; col += 32) {
        const uint32_t n = r * d.cols + col;
        const bool free_ = !((bits[n >> 5] >> (n & 31)) & 1u);
        const uint32_t colour = (r + col) & 1u;
        cnt0 += free_ && colour == 0;
        cnt1 += free_ && colour == 1;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        cnt0 += __shfl_xor_sync(0xFFFFFFFFu, cnt0, o);
        cnt1 += __shfl_xor_sync(0xFFFFFFFFu, cnt1, o);
    }
    if (lane == 0) {
        d.rowstart[((size_t)g * 2 + 0) * (d.rows + 1) + r] = cnt0;
        d.rowstart[((size_t)g * 2 + 1) * (d.rows + 1) + r] = cnt1;
    }
}

// one warp per (grid, colour): exclusive scan of the row counts in place
__global__ void k_rowscan(Dev d)
{
    const int g = blockIdx.x, colour = blockIdx.y;
    const uint32_t lane = threadIdx.x;
    uint32_t* rs = d.rowstart + ((size_t)g * 2 + colour) * (d.rows + 1);
    uint32_t carry = 0;
    for (uint32_t base = 0; base < (uint32_t)d.rows; base += 32) {
        const uint32_t r = base + lane;
        const uint32_t c = r < (uint32_t)d.rows ? rs[r] : 0u;
        uint32_t x = c;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t y = __shfl_up_sync(0xFFFFFFFFu, x, o);
            if (lane >= (uint32_t)o) x += y;
        }
        if (r < (uint32_t)d.rows) rs[r] = carry + x - c;
        carry += __shfl_sync(0xFFFFFFFFu, x, 31);
    }
    if (lane == 0) {
        rs[d.rows] = carry;
        d.states[g].n_free[colour] = carry;
        uint32_t* list = d.lists + ((size_t)g * 2 + colour) * d.LC;
        list[carry] = LIST_SENTINEL;            // pads an odd count to a whole pair
        list[carry + 1] = LIST_SENTINEL;
    }
}

__global__ void __launch_bounds__(256) k_build_lists(Dev d)
{
    const int g = blockIdx.y;
    const uint32_t r = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const uint32_t lane = threadIdx.x & 31;
    if (r >= (uint32_t)d.rows) return;
    const uint32_t* bits = d.bits + (size_t)g * d.words;
    for (uint32_t colour = 0; colour < 2; ++colour) {
        const uint32_t par = (r + colour) & 1u;                         // parity of this colour's columns in row r
        uint32_t pos = d.rowstart[((size_t)g * 2 + colour) * (d.rows + 1) + r];
        uint32_t* list = d.lists + ((size_t)g * 2 + colour) * d.LC;
        for (uint32_t j0 = 0; j0 < d.W; j0 += 32) {
            const uint32_t j = j0 + lane, col = 2u * j + par;
            bool free_ = false;
            if (col < (uint32_t)d.cols) {
                const uint32_t n = r * d.cols + col;
                free_ = !((bits[n >> 5] >> (n & 31)) & 1u);
            }
            const uint32_t b = __ballot_sync(0xFFFFFFFFu, free_);
            if (free_) list[pos + __popc(b & ((1u << lane) - 1u))] = padded_index(r, col, d.Wp) | (par << 31);
            pos += __popc(b);
        }
    }
}

// ---------------------------------------------------------------------------
// a2  tile frames.  The grid is cut into TR x TC core tiles; a tile's frame is
// its core plus a halo of H sites on every side.  For each tile the free
// sites of the frame with ring < H (ring = Chebyshev distance outside the
// core, 0 inside) are listed per colour, outermost ring first, so that the
// sites a half-sweep of a K-sweep pass still needs are a suffix of the list.
// ---------------------------------------------------------------------------
struct TileGeom { int r0, c0, TRc, TCc; };

__device__ __forceinline__ TileGeom tile_geom(const Dev& d, int tile)
{
    TileGeom t;
    const int ty = tile / d.ntx, tx = tile - ty * d.ntx;
    t.r0 = ty * d.TR; t.c0 = tx * d.TC;
    t.TRc = min(d.TR, d.rows - t.r0); t.TCc = min(d.TC, d.cols - t.c0);
    return t;
}

// class of frame site (lr, lc): returns false if outside the grid, fixed, or on the outermost ring
__device__ __forceinline__ bool frame_site_class(const Dev& d, const uint32_t* __restrict__ bits, const TileGeom& t,
                                                 int lr, int lc, int& colour, int& ring)
{
    const int r = t.r0 - d.H + lr, col = t.c0 - d.H + lc;
    if (r < 0 || r >= d.rows || col < 0 || col >= d.cols) return false;
    const uint32_t n = (uint32_t)r * d.cols + col;
    if ((bits[n >> 5] >> (n & 31)) & 1u) return false;
    const int dr = max(max(d.H - lr, lr - (d.H + t.TRc - 1)), 0);
    const int dc = max(max(d.H - lc, lc - (d.H + t.TCc - 1)), 0);
    ring = max(dr, dc);
    colour = (r + col) & 1;
    return ring < d.H;
}

__global__ void __launch_bounds__(256) k_tile_count(Dev d)
{
    const int tile = blockIdx.x, g = blockIdx.y;
    __shared__ uint32_t hist[2][MAX_H + 1];
    for (int i = threadIdx.x; i < 2 * (MAX_H + 1); i += blockDim.x) (&hist[0][0])[i] = 0;
    __syncthreads();
    const TileGeom t = tile_geom(d, tile);
    const uint32_t* bits = d.bits + (size_t)g * d.words;
    for (int i = threadIdx.x; i < d.FR * d.FC; i += blockDim.x) {
        const int lr = i / d.FC, lc = i - lr * d.FC;
        int colour, ring;
        if (frame_site_class(d, bits, t, lr, lc, colour, ring)) atomicAdd(&hist[colour][ring], 1u);
    }
    __syncthreads();
    if (threadIdx.x < 2) {
        TileMeta& m = d.tile_meta[(size_t)g * d.ntiles + tile];
        const int c = threadIdx.x;
        uint32_t run = 0;
        for (int k = MAX_H; k >= 0; --k) { run += hist[c][k]; m.cge[c][k] = run; }
    }
}

// one warp per grid: exclusive scan of the tiles' entry counts, and their maximum
__global__ void k_tile_scan(Dev d)
{
    const int g = blockIdx.x;
    const uint32_t lane = threadIdx.x;
    TileMeta* m = d.tile_meta + (size_t)g * d.ntiles;
    uint32_t carry = 0, mx = 0;
    for (int base = 0; base < d.ntiles; base += 32) {
        const int i = base + lane;
        const uint32_t c = i < d.ntiles ? m[i].cge[0][0] + m[i].cge[1][0] : 0u;
        mx = max(mx, c);
        uint32_t x = c;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t y = __shfl_up_sync(0xFFFFFFFFu, x, o);
            if (lane >= (uint32_t)o) x += y;
        }
        if (i < d.ntiles) m[i].base = carry + x - c;
        carry += __shfl_sync(0xFFFFFFFFu, x, 31);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) mx = max(mx, __shfl_xor_sync(0xFFFFFFFFu, mx, o));
    if (lane == 0) d.states[g].max_tile_entries = mx;
}

__global__ void __launch_bounds__(256) k_tile_fill(Dev d)
{
    const int tile = blockIdx.x, g = blockIdx.y;
    __shared__ uint32_t cursor[2][MAX_H + 1];
    for (int i = threadIdx.x; i < 2 * (MAX_H + 1); i += blockDim.x) (&cursor[0][0])[i] = 0;
    __syncthreads();
    const TileGeom t = tile_geom(d, tile);
    const TileMeta& m = d.tile_meta[(size_t)g * d.ntiles + tile];
    const uint32_t* bits = d.bits + (size_t)g * d.words;
    uint32_t* out = d.entries + (size_t)g * d.entry_stride + m.base;
    for (int i = threadIdx.x; i < d.FR * d.FC; i += blockDim.x) {
        const int lr = i / d.FC, lc = i - lr * d.FC;
        int colour, ring;
        if (frame_site_class(d, bits, t, lr, lc, colour, ring)) {
            // colour 0 first; within a colour the rings in descending order
            const uint32_t pos = (colour ? m.cge[0][0] : 0u) + m.cge[colour][ring + 1] + atomicAdd(&cursor[colour][ring], 1u);
            out[pos] = (uint32_t)i | ((uint32_t)lr << 16);
        }
    }
}

// ---------------------------------------------------------------------------
// a2  initial state (Alg. 2 step 2.2, L176): phi ~ U(0, 2 pi) at prediction
// sites from the INIT stream; every site's unit vector (cos q phi, sin q phi)
// into BOTH vector buffers (sample sites are never written again).
// ---------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_init_state(Dev d)
{
    const int g = blockIdx.y;
    const uint32_t n = blockIdx.x * blockDim.x + threadIdx.x;
    if (n >= d.N) return;
    const size_t o = (size_t)g * d.N + n;
    const bool fixed = (d.bits[(size_t)g * d.words + (n >> 5)] >> (n & 31)) & 1u;
    float p;
    if (fixed) p = d.phi[o];
    else {
        const uint4 x = philox4x32_10(n >> 2, 0u, 0u, (uint32_t)g, d.key0, d.key1);
        const uint32_t w = (n & 3u) == 0 ? x.x : (n & 3u) == 1 ? x.y : (n & 3u) == 2 ? x.z : x.w;
        p = __fmul_rn(TWO_PI_F, u01(w));
        d.phi[o] = p;
    }
    const uint32_t r = n / d.cols, col = n - r * d.cols;
    float sn, cs;
    sincosf(__fmul_rn(d.q, p), &sn, &cs);
    const size_t at = (size_t)((r + col) & 1u) * d.VS + padded_index(r, col, d.Wp);
    cur_vec(d, g, 0)[at] = make_float2(cs, sn);
    cur_vec(d, g, 1)[at] = make_float2(cs, sn);
}

// ---------------------------------------------------------------------------
// a3  UPDATE of one prediction site (Alg. 1) in vector form.
// v = (cos q phi, sin q phi); (hx, hy) = (C, S) = sum over the neighbours.
// ---------------------------------------------------------------------------
template <bool QHALF, int ORMODE>
__device__ __forceinline__ float2 update_site(float2 v, float hx, float hy, float2 n_up, float2 n_dn, float2 n_lf,
                                              float2 n_rt, float uc, float r, float hd_scale, float nlT,
                                              float bc, float bs, bool renorm, uint32_t& accepted)
{
    float px = v.x, py = v.y;
    // Alg. 1 line 1: over-relaxation.  Reflect v about h: q phi' = 2 Theta - q phi keeps h.v,
    // i.e. the local energy (L156, L265; R2).  Out of [0, 2 pi]: keep the spin.
    if (ORMODE == 0) {
        const float R2 = fmaf(hx, hx, hy * hy);
        const float k = __fdividef(2.0f * fmaf(px, hx, py * hy), R2);   // 0/0 -> NaN -> kept below
        const float fx = fmaf(k, hx, -px), fy = fmaf(k, hy, -py);
        // Theta = atan2(S, C) < 0 when S < 0 (only through sin(q * TWO_PI_F) = -8.7e-8 of a sample at the
        // data maximum, with the other neighbours cancelling): then q phi' = 2 Theta - q phi < 0, out of range (R17)
        bool in = fy >= 0.0f && hy >= 0.0f;
        if (!QHALF) in = in && (fmaf(fx, bs, -fy * bc) >= 0.0f);
        px = in ? fx : px; py = in ? fy : py;
    } else if (ORMODE == 1) {
        // Eq. 6 as printed (L158), q = 1/2 only: phi' = [2 atan2(sum sin phi_j, sum cos phi_j) - phi] mod 2 pi,
        // with cos phi_j = c^2 - s^2, sin phi_j = 2 c s; q phi' = Theta_1 - q phi (mod pi)
        const float C1 = (n_up.x * n_up.x - n_up.y * n_up.y) + (n_dn.x * n_dn.x - n_dn.y * n_dn.y)
                       + (n_lf.x * n_lf.x - n_lf.y * n_lf.y) + (n_rt.x * n_rt.x - n_rt.y * n_rt.y);
        const float S1 = 2.0f * (n_up.x * n_up.y + n_dn.x * n_dn.y + n_lf.x * n_lf.y + n_rt.x * n_rt.y);
        const float R2 = fmaf(C1, C1, S1 * S1);
        const float inv = R2 > 0.0f ? rsqrtf(R2) : 0.0f;
        const float ex = R2 > 0.0f ? C1 * inv : 1.0f, ey = S1 * inv;      // atan2(0,0) = 0
        float fx = fmaf(ex, px, ey * py), fy = fmaf(ey, px, -ex * py);
        if (fy < 0.0f) { fx = -fx; fy = -fy; }
        px = fx; py = fy;
    }
    // lines 2-3: phi'' = phi' + 2 pi (u - 1/2)/a (mod 2 pi): rotate by d = q delta = 2 hd
    const float hd = uc * hd_scale;
    float sh, ch;
    sincos_small(hd, sh, ch);
    const float sd = 2.0f * sh * ch, omc = 2.0f * sh * sh;               // sin d, 1 - cos d
    float rx = px - fmaf(omc, px, sd * py);
    float ry = py - fmaf(omc, py, -sd * px);
    // line 4: dH = -h.(v'' - v') = (1 - cos d)(h.v') + sin d (h x v'): no cancellation at low T
    const float hdotp = fmaf(hx, px, hy * py);
    const float hcrossp = fmaf(hx, py, -hy * px);
    float dH = fmaf(omc, hdotp, sd * hcrossp);
    if (QHALF) {
        // q = 1/2: q phi in [0, pi]; leaving it <=> sin < 0; phi -/+ 2 pi <=> v -> -v
        if (ry < 0.0f) { rx = -rx; ry = -ry; dH = fmaf(2.0f, hdotp, -dH); }
    } else {
        const bool under = hd < 0.0f && ry < 0.0f;
        const bool over = hd > 0.0f && !(ry >= 0.0f && fmaf(rx, bs, -ry * bc) >= 0.0f);
        if (under || over) {
            const float s2 = under ? bs : -bs;
            const float wx = fmaf(rx, bc, -ry * s2), wy = fmaf(rx, s2, ry * bc);
            rx = wx; ry = wy;
            dH = hdotp - fmaf(hx, rx, hy * ry);
        }
    }
    // lines 5-6: AP = min{1, exp(-dH/T)}; accept phi'' if AP > r else keep phi'
    const bool acc = dH <= 0.0f || ex2_approx(dH * nlT) > r;
    accepted += acc;
    float nx = acc ? rx : px, ny = acc ? ry : py;
    if (renorm) {   // keep |v| = 1 against rounding drift (first-order Newton step of 1/|v|), once per pass
        const float sc = fmaf(-0.5f, fmaf(nx, nx, ny * ny), 1.5f);
        nx *= sc; ny *= sc;
    }
    return make_float2(nx, ny);
}

// ---------------------------------------------------------------------------
// a3/a4  the hot kernel: K whole sweeps (colour 0 then colour 1, L261-265) of
// one tile, on a copy of its frame in shared memory (temporal blocking).
// Reads the state from one vector buffer and writes the tile's core to the
// other, so tiles of one launch never see each other's writes.  Sites of the
// halo are updated redundantly; they reproduce the neighbouring tiles'
// results bit for bit because the random numbers are keyed by (site, sweep).
// After half-sweep number hs (0-based) the frame is valid up to ring
// 2K-1-hs, so each half-sweep only updates the suffix of the entry list
// with ring <= 2K-1-hs.  Optionally fused at the end of the pass:
//   PASS_ENERGY      a5: - sum over the core's colour-1 sites of v.h (each bond once)
//   PASS_COUNT       a5: accepted proposals of the core sites
//   PASS_ACCUMULATE  a7: acc += phi at the core's prediction sites
// ---------------------------------------------------------------------------
template <bool QHALF, int ORMODE>
__global__ void __launch_bounds__(TILE_THREADS, 2) k_tilepass(Dev d, uint32_t K, uint32_t t_off, uint32_t flip, uint32_t flags)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ uint32_t s_cge[2][MAX_H + 1];
    __shared__ uint32_t s_accepted;
    __shared__ double s_red[TILE_THREADS / 32];

    const int tile = blockIdx.x, g = blockIdx.y;
    const GridState& st = d.states[g];
    if ((flags & PASS_CHECK_DONE) && st.done) return;

    float2*   S  = reinterpret_cast<float2*>(smem_raw);
    uint32_t* E  = reinterpret_cast<uint32_t*>(S + d.FR * d.FC);
    uint2*    SP = reinterpret_cast<uint2*>(E + d.max_entries);

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    constexpr int NW = TILE_THREADS / 32;
    const TileGeom tg = tile_geom(d, tile);
    const TileMeta& meta = d.tile_meta[(size_t)g * d.ntiles + tile];
    const int H = d.H, FC = d.FC;
    const int X = min((int)(2 * K), H);                      // rings of the frame this pass needs
    const uint32_t src_buf = st.cur ^ flip;
    const float2* src = cur_vec(d, g, src_buf);
    float2*       dst = cur_vec(d, g, src_buf ^ 1u);

    if (tid < 2 * (MAX_H + 1)) (&s_cge[0][0])[tid] = (&meta.cge[0][0])[tid];
    if (tid == 0) s_accepted = 0;
    const uint32_t nE = meta.cge[0][0] + meta.cge[1][0];
    {
        const uint32_t* gE = d.entries + (size_t)g * d.entry_stride + meta.base;
        for (uint32_t i = tid; i < nE; i += TILE_THREADS) E[i] = gE[i];
    }
    // frame load: out-of-grid sites are zero vectors = open boundary
    for (int lr = H - X + warp; lr < H + tg.TRc + X; lr += NW) {
        const int r = tg.r0 - H + lr;
        const bool rin = r >= 0 && r < d.rows;
        for (int lc = H - X + lane; lc < H + tg.TCc + X; lc += 32) {
            const int col = tg.c0 - H + lc;
            float2 v = make_float2(0.0f, 0.0f);
            if (rin && col >= 0 && col < d.cols)
                v = src[(size_t)((r + col) & 1) * d.VS + (uint32_t)(r + 1) * d.Wp + (uint32_t)(col >> 1) + 1u];
            S[lr * FC + lc] = v;
        }
    }
    __syncthreads();

    const float hs = st.hd_scale, nlT = st.neg_log2e_over_T;
    const uint32_t t0 = st.t + t_off;
    const int nbase = (tg.r0 - H) * d.cols + (tg.c0 - H), ncorr = d.cols - FC;
    const bool count = flags & PASS_COUNT;
    uint32_t accepted = 0;

    for (uint32_t s = 0; s < K; ++s) {
        const uint32_t t = t0 + s;
        const bool odd = t & 1u;
        const bool fresh = !odd || s == 0 || !d.use_spare;           // draw a new Philox block for (site, t >> 1)
        const bool stash = d.use_spare && !odd && s + 1 < K;        // keep words 2,3 for sweep t + 1
        const bool renorm = s + 1 == K;
#pragma unroll 1
        for (int c = 0; c < 2; ++c) {
            const int R = (int)(2 * K) - 1 - (int)(2 * s + c);       // rings still needed
            const uint32_t first = R + 1 <= MAX_H ? s_cge[c][R + 1] : 0u;
            const uint32_t last = s_cge[c][0], core_from = s_cge[c][1];
            const uint32_t base = c ? s_cge[0][0] : 0u;
            for (uint32_t e = first + tid; e < last; e += TILE_THREADS) {
                const uint32_t ent = E[base + e];
                const uint32_t off = ent & 0xFFFFu, lr = ent >> 16;
                const float2 v = S[off], up = S[off - FC], dn = S[off + FC], lf = S[off - 1], rt = S[off + 1];
                uint32_t w0, w1;
                if (fresh) {
                    const uint32_t n = (uint32_t)(nbase + (int)off + (int)lr * ncorr);
                    const uint4 x = philox4x32_10(n, t >> 1, 2u, (uint32_t)g, d.key0, d.key1);
                    w0 = odd ? x.z : x.x; w1 = odd ? x.w : x.y;
                    if (stash) SP[base + e] = make_uint2(x.z, x.w);
                } else {
                    const uint2 sp = SP[base + e];
                    w0 = sp.x; w1 = sp.y;
                }
                const float hx = (up.x + dn.x) + (lf.x + rt.x), hy = (up.y + dn.y) + (lf.y + rt.y);
                uint32_t a = 0;
                S[off] = update_site<QHALF, ORMODE>(v, hx, hy, up, dn, lf, rt, u01_centered(w0), u01(w1), hs, nlT,
                                                    d.bc, d.bs, renorm, a);
                if (count && e >= core_from) accepted += a;
            }
            __syncthreads();
        }
    }

    // write the core back (both colours, whole rows: coalesced in each colour plane)
    for (int lr = H + warp; lr < H + tg.TRc; lr += NW) {
        const int r = tg.r0 - H + lr;
        for (int lc = H + lane; lc < H + tg.TCc; lc += 32) {
            const int col = tg.c0 - H + lc;
            dst[(size_t)((r + col) & 1) * d.VS + (uint32_t)(r + 1) * d.Wp + (uint32_t)(col >> 1) + 1u] = S[lr * FC + lc];
        }
    }
    if (flags & PASS_ACCUMULATE) {
        // a7 (Alg. 2 step 6, L207-211): acc += phi at the core's prediction sites
        for (int c = 0; c < 2; ++c) {
            const uint32_t base = c ? s_cge[0][0] : 0u;
            float* acc = d.acc + ((size_t)g * 2 + c) * d.VS;
            for (uint32_t e = s_cge[c][1] + tid; e < s_cge[c][0]; e += TILE_THREADS) {
                const uint32_t ent = E[base + e];
                const uint32_t off = ent & 0xFFFFu, lr = ent >> 16, lc = off - lr * FC;
                const int r = tg.r0 - H + (int)lr, col = tg.c0 - H + (int)lc;
                acc[(uint32_t)(r + 1) * d.Wp + (uint32_t)(col >> 1) + 1u] += angle_of(S[off], d.inv_q);
            }
        }
    }
    if (count) {
        accepted = __reduce_add_sync(0xFFFFFFFFu, accepted);
        if (lane == 0 && accepted) atomicAdd(&s_accepted, accepted);
    }
    if (flags & PASS_ENERGY) {
        // a5: H_tile = - sum over the core's colour-1 sites (fixed ones too) of v . h; fixed summation order
        double sum = 0.0;
        for (int lr = H + warp; lr < H + tg.TRc; lr += NW) {
            const int r = tg.r0 - H + lr;
            float row = 0.0f;
            // first colour-1 column of this row at or after the core's first column
            for (int lc = H + ((r + tg.c0 + 1) & 1) + 2 * lane; lc < H + tg.TCc; lc += 64) {
                const int off = lr * FC + lc;
                const float2 v = S[off], up = S[off - FC], dn = S[off + FC], lf = S[off - 1], rt = S[off + 1];
                row += fmaf(v.x, (up.x + dn.x) + (lf.x + rt.x), v.y * ((up.y + dn.y) + (lf.y + rt.y)));
            }
            sum += (double)row;
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) sum += __shfl_xor_sync(0xFFFFFFFFu, sum, o);
        if (lane == 0) s_red[warp] = sum;
    }
    __syncthreads();
    if (tid == 0) {
        if (count && s_accepted) atomicAdd(&d.states[g].accepted, (unsigned long long)s_accepted);
        if (flags & PASS_ENERGY) {
            double s = 0.0;
            for (int w = 0; w < NW; ++w) s += s_red[w];
            d.e_partials[(size_t)g * d.n_partials + tile] = -s;
        }
    }
}

// ---------------------------------------------------------------------------
// a5  energy of the current state on demand (mpr_energy): H = - sum over the
// colour-1 sites i of v_i . h_i (every bond joins the two colours; Eq. 2).
// Fixed block count and a fixed summation tree: bitwise reproducible.
// ---------------------------------------------------------------------------
__global__ void __launch_bounds__(ENERGY_THREADS) k_energy(Dev d)
{
    const int g = blockIdx.y;
    __shared__ double warp_sum[ENERGY_THREADS / 32];
    const float2* own = cur_vec(d, g, d.states[g].cur) + d.VS;
    const float2* oth = cur_vec(d, g, d.states[g].cur);
    double sum = 0.0;
    for (uint32_t r = blockIdx.x; r < (uint32_t)d.rows; r += gridDim.x) {
        const uint32_t par = (r + 1u) & 1u;
        float row = 0.0f;
        int cnt = 0;
        for (uint32_t j = threadIdx.x; j < d.W; j += ENERGY_THREADS) {
            const uint32_t li = (r + 1u) * d.Wp + j + 1u;
            const float2 v = own[li];
            const float2 up = oth[li - d.Wp], dn = oth[li + d.Wp], lf = oth[li - 1u + par], rt = oth[li + par];
            const float hx = (up.x + dn.x) + (lf.x + rt.x), hy = (up.y + dn.y) + (lf.y + rt.y);
            row += fmaf(v.x, hx, v.y * hy);
            if (++cnt == 8) { sum += (double)row; row = 0.0f; cnt = 0; }
        }
        sum += (double)row;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) sum += __shfl_xor_sync(0xFFFFFFFFu, sum, o);
    if ((threadIdx.x & 31) == 0) warp_sum[threadIdx.x >> 5] = sum;
    __syncthreads();
    if (threadIdx.x == 0) {
        double s = 0.0;
        for (int w = 0; w < ENERGY_THREADS / 32; ++w) s += warp_sum[w];
        d.e_partials[(size_t)g * d.n_partials + blockIdx.x] = -s;
    }
}

__device__ __forceinline__ double sum_energy_partials(const Dev& d, int g, int n)
{
    const double* p = d.e_partials + (size_t)g * d.n_partials;
    double s = 0.0;
    for (int b = threadIdx.x; b < n; b += 32) s += p[b];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xFFFFFFFFu, s, o);
    return s;
}

__global__ void k_energy_query(Dev d, int n_partials)
{
    const int g = blockIdx.x;
    const double H = sum_energy_partials(d, g, n_partials);
    if (threadIdx.x == 0) d.states[g].e_query = H / d.n_bonds;
}

// ---------------------------------------------------------------------------
// a6  equilibration controller: Alg. 2 steps 5.2-5.5 for
// one grid per warp, after the sweep (5.1) with its fused energy reduction.
// Commits the sweep: t += 1 and the vector buffers swap roles.
// ---------------------------------------------------------------------------
__global__ void k_controller(Dev d)
{
    const int g = blockIdx.x;
    GridState& s = d.states[g];
    if (s.done) return;
    const double H = sum_energy_partials(d, g, d.ntiles);
    if (threadIdx.x != 0) return;
    const uint32_t i = s.i;
    const double P = (double)s.n_free[0] + (double)s.n_free[1];
    // 5.2 acceptance control: a(i+1) = 1 + (i+1)/k_a while A < A_targ
    const double A = (double)s.accepted / P;
    double a = s.a;
    if (A < d.A_targ) a = 1.0 + (double)(i + 1u) / d.k_a;
    // 5.3 e(i+1) = H / N_GP
    const double e = H / d.n_bonds;
    s.e_ring[(i + 1u) % d.n_fit] = e;
    // 5.4 slope of the last n_fit energies e(i+2-n_fit) .. e(i+1): degree-1 Savitzky-Golay = OLS (R9)
    double k = s.k;
    if (i >= d.n_fit && i % d.n_f == 0) {
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
    // 5.5
    s.i = i + 1u; s.t += 1u; s.cur ^= 1u; s.a = a; s.k = k; s.A_last = A; s.e_last = e; s.accepted = 0ull;
    s.hd_scale = (float)((double)d.q * (0.5 * (double)TWO_PI_F) / a);
    if (!(k < 0.0 && i + 1u < d.equil_cap)) { s.done = 1u; d.done_flags[g] = 1u; }
}

// scalar state edits ---------------------------------------------------------
// mode 0: a <- a_value for every grid; mode 1: keep a (refresh the derived scale only)
__global__ void k_set_a(Dev d, int mode, double a_value, int zero_accepted)
{
    const int g = blockIdx.x * blockDim.x + threadIdx.x;
    if (g >= d.batch) return;
    GridState& s = d.states[g];
    if (mode == 0) s.a = a_value;
    s.hd_scale = (float)((double)d.q * (0.5 * (double)TWO_PI_F) / s.a);
    if (zero_accepted) s.accepted = 0ull;
}
// commit passes that ran with (t_off, flip) arguments: t += n_sweeps, swap buffers if the pass count was odd
__global__ void k_commit(Dev d, uint32_t n_sweeps, uint32_t flip, uint32_t n_realizations)
{
    const int g = blockIdx.x * blockDim.x + threadIdx.x;
    if (g >= d.batch) return;
    GridState& s = d.states[g];
    s.t += n_sweeps; s.cur ^= flip; s.realizations += n_realizations;
}
__global__ void k_set_t(Dev d, uint32_t t)
{
    const int g = blockIdx.x * blockDim.x + threadIdx.x;
    if (g < d.batch) d.states[g].t = t;
}
__global__ void k_begin_run(Dev d, const float* __restrict__ T)
{
    const int g = blockIdx.x * blockDim.x + threadIdx.x;
    if (g >= d.batch) return;
    GridState& s = d.states[g];
    s.t = 0; s.done = 0; s.cur = 0; s.i = 0; s.realizations = 0; s.accepted = 0ull;
    s.a = 1.0; s.k = -1.0; s.A_last = 0.0; s.e_last = 0.0;
    s.T = (double)T[g];
    s.neg_log2e_over_T = (float)(-1.4426950408889634 / (double)T[g]);
    s.hd_scale = (float)((double)d.q * (0.5 * (double)TWO_PI_F));
    d.done_flags[g] = 0;
}

// ---------------------------------------------------------------------------
// a8  prediction (Alg. 2 step 7, L148, L212) at the free sites; the caller
// has already copied the input values (sample sites bit for bit) into out.
// ---------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_predict(Dev d, float* __restrict__ out)
{
    const int g = blockIdx.y, colour = blockIdx.z;
    const uint32_t o = blockIdx.x * blockDim.x + threadIdx.x;
    const GridState& s = d.states[g];
    if (o >= s.n_free[colour]) return;
    const uint32_t idx = d.lists[((size_t)g * 2 + colour) * d.LC + o], li = idx & 0x7FFFFFFFu, par = idx >> 31;
    const uint32_t r = li / d.Wp - 1u, col = 2u * (li - (r + 1u) * d.Wp - 1u) + par;
    const double mean_phi = (double)d.acc[((size_t)g * 2 + colour) * d.VS + li] / (double)s.realizations;
    const double z = (double)s.zmin + mean_phi * ((double)s.zmax - (double)s.zmin) / (double)TWO_PI_F;
    out[(size_t)g * d.N + (size_t)r * d.cols + col] = (float)z;
}

// angle import / export at the free sites -----------------------------------
__global__ void __launch_bounds__(256) k_export_angles(Dev d)
{
    const int g = blockIdx.y, colour = blockIdx.z;
    const uint32_t o = blockIdx.x * blockDim.x + threadIdx.x;
    if (o >= d.states[g].n_free[colour]) return;
    const uint32_t idx = d.lists[((size_t)g * 2 + colour) * d.LC + o], li = idx & 0x7FFFFFFFu, par = idx >> 31;
    const uint32_t r = li / d.Wp - 1u, col = 2u * (li - (r + 1u) * d.Wp - 1u) + par;
    const float2 v = cur_vec(d, g, d.states[g].cur)[(size_t)colour * d.VS + li];
    d.phi[(size_t)g * d.N + (size_t)r * d.cols + col] = angle_of(v, d.inv_q);
}
__global__ void __launch_bounds__(256) k_import_angles(Dev d, const float* __restrict__ phi_in)
{
    const int g = blockIdx.y, colour = blockIdx.z;
    const uint32_t o = blockIdx.x * blockDim.x + threadIdx.x;
    if (o >= d.states[g].n_free[colour]) return;
    const uint32_t idx = d.lists[((size_t)g * 2 + colour) * d.LC + o], li = idx & 0x7FFFFFFFu, par = idx >> 31;
    const uint32_t r = li / d.Wp - 1u, col = 2u * (li - (r + 1u) * d.Wp - 1u) + par;
    const size_t n = (size_t)g * d.N + (size_t)r * d.cols + col;
    float p = phi_in[n];
    p = p < 0.0f ? 0.0f : p;
    p = p > TWO_PI_F ? TWO_PI_F : p;
    d.phi[n] = p;
    float sn, cs;
    sincosf(__fmul_rn(d.q, p), &sn, &cs);
    cur_vec(d, g, d.states[g].cur)[(size_t)colour * d.VS + li] = make_float2(cs, sn);
}

}  // namespace mpr
