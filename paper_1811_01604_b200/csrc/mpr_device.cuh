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
#include <cuda.h>
#include <cuda_runtime.h>
// -DMPR_CHECKED (build.build_checked(): libmpr_b200_checked.so): bounds checks of every shared-memory and accumulator
// index of the tile pass as device-side assertions.  compute-sanitizer is closed on the GPU pool this was developed
// on (profiles/r02d); tests/sanitizer_driver.py --lib <checked library> runs every kernel family through them.
#ifdef MPR_CHECKED
#include <cassert>
#define MPR_CHECK(cond) assert(cond)
#else
#define MPR_CHECK(cond) ((void)0)
#endif

namespace mpr {

constexpr float    TWO_PI_F       = 6.28318530717958647692f;  // float nearest 2 pi; state space [0, TWO_PI_F]
constexpr int      MAX_NFIT       = 256;
constexpr int      TILE_THREADS   = 256;                      // threads of a tile pass CTA
constexpr int      MAX_H          = 16;                       // largest halo: up to 8 sweeps per tile pass
constexpr int      STD_FC         = 82;                       // frame pitch of the standard 64 x 64 tile with halo 8 (compile-time in k_tilepass)
constexpr int      ENERGY_BLOCKS  = 592;                      // 4 x 148 SMs; fixed so the sum order is deterministic
constexpr int      ENERGY_THREADS = 256;
constexpr int      PHILOX_ROUNDS  = 10;

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
    double   e_query;            // result slot of mpr_energy / mpr_sample_energy
    double   e_sum;              // mpr_measure_energy: sum over the measured sweeps of e
    uint32_t n_meas;             //   and their number
    unsigned long long n_pairs;  // N_SP of Eq. 4 (mpr_sample_energy)
    double   e_ring[MAX_NFIT];   // e(i) at slot i % n_fit
};

// Free sites of one tile frame (core + halo), see k_tile_fill.
struct TileMeta {
    uint32_t cle[2][MAX_H];           // cle[c][k] = entries of colour c with ring <= k (ring = distance outside the core)
};
// colour 1's list starts on a 16-entry boundary after colour 0's
__host__ __device__ __forceinline__ uint32_t colour1_base(uint32_t n0) { return (n0 + 15u) & ~15u; }

// Device view of one context (passed by value to kernels).
struct Dev {
    GridState* states;         // [nv]
    uint32_t*  done_flags;     // [batch] copy of GridState::done for cheap host polling
    double*    e_partials;     // [batch][n_partials]
    float*     values;         // [batch][N] verbatim copy of the input values
    float*     phi;            // [batch][N] angle view: Eq. 1 at sample sites (never rewritten), export buffer at free sites
    uint32_t*  bits;           // [batch][words] fixed-site bitmask
    float2*    vec;            // [2 buffers][nv][rows][pitch] row-major unit vectors (pitch = cols rounded up to even)
    float*     acc;            // [nv][ntiles][acc_stride] sum over realizations of phi at the prediction sites, per tile in the
                               // order of the tile's CORE entries: colour 0's at 0.., colour 1's from colour1_base(count of colour 0)
    float*     m2;             // same shape: sum of squared deviations from the running mean (Welford), for the spread (L212)
    TileMeta*  tile_meta;      // [batch][ntiles]
    uint16_t*  entries;        // [batch][entry_stride] tile frames' free sites: offset in the frame (row * FC + col)
    int        batch, rows, cols;   // batch = grids with data of their own
    int        chains, nv;          // chains per grid (reading R25) and nv = batch * chains states: chain c of grid g is
                                    // state v = g + c * batch; it shares grid g's values, mask and tile lists
    uint32_t   N, words, pitch;
    size_t     VG;             // float2 elements of one grid in one buffer = rows * pitch
    size_t     VB;             // float2 elements per vector buffer = nv * VG
    size_t     entry_stride;   // entries per grid = ntiles * tile_entries
    uint32_t   tile_entries;   // room of one tile's lists (worst case: every frame site free), multiple of 16; tile i's
                               // lists start at i * tile_entries, so that loading them needs nothing read first
    uint32_t   n_partials;
    uint32_t   acc_stride;     // floats of one tile's accumulators: TR * TC rounded up to 16, + 16
    // row-block decomposition of one grid over several contexts (mpr_create_slab): this context's grid is rows
    // [slab_row0, slab_row0 + rows) of a larger one; its rows [own_r0, own_r1) are its own, the others are ghost copies
    // of the neighbouring slabs' rows.  A plain context: site_off = 0, own_r0 = 0, own_r1 = rows.
    uint32_t   site_off;       // slab_row0 * cols: added to row * cols + col, the site word of the Philox counter
    int        own_r0, own_r1; // rows counted in the energy, the accepted proposals and the number of prediction sites
    // tiling
    int        TR, TC, H, FR, FC, ntx, nty, ntiles;
    uint32_t   max_entries;    // shared-memory capacity for entries (multiple of 8)
    uint32_t   fc_inv;         // ceil(2^24 / FC): frame row of offset o = (o * fc_inv) >> 24, exact for o < 2^16
    int        use_spare;      // keep the odd sweep's random words in shared memory
    uint32_t   rk0[PHILOX_ROUNDS], rk1[PHILOX_ROUNDS];   // Philox round keys: (seed lo, seed hi) + r * Weyl constants
    float      q, inv_q;
    float      bc, bs;         // (cos 2 pi q, sin 2 pi q): upper end of the q*phi range
    // Alg. 2 controller constants
    uint32_t   n_f, n_fit, equil_cap;
    int        burn_in_only;   // unconditional context: no slope stop
    double     A_targ, k_a, n_bonds;
};

__device__ __forceinline__ float2* vec_grid(const Dev& d, int g, uint32_t which)
{
    return d.vec + (size_t)which * d.VB + (size_t)g * d.VG;
}

// ---------------------------------------------------------------------------
// Philox4x32-10 (Salmon et al., SC'11), the generator PAPER.md L267 names.
// The ten round keys are precomputed on the host (Dev::rk0 / rk1).
// ---------------------------------------------------------------------------
__device__ __forceinline__ uint4 philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                               const uint32_t (&rk0)[PHILOX_ROUNDS], const uint32_t (&rk1)[PHILOX_ROUNDS])
{
#pragma unroll
    for (int r = 0; r < PHILOX_ROUNDS; ++r) {
        const uint64_t p0 = (uint64_t)c0 * 0xD2511F53u;     // IMAD.WIDE: hi and lo in one instruction
        const uint64_t p1 = (uint64_t)c2 * 0xCD9E8D57u;
        const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ rk0[r];
        const uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ rk1[r];
        c0 = n0; c1 = (uint32_t)p1; c2 = n2; c3 = (uint32_t)p0;
    }
    return make_uint4(c0, c1, c2, c3);
}

// Uniform u = (2 (x >> 9) + 1) 2^-24 in (0,1) (R13), built without
// an integer->float conversion: f = 1.m in [1,2) with m = x >> 9, so
// u = f - (1 - 2^-24), exact in one subtraction ((2m+1) 2^-24 has 24 bits).
__device__ __forceinline__ float one_plus_m(uint32_t x) { return __uint_as_float(0x3F800000u | (x >> 9)); }
__device__ __forceinline__ float u01(uint32_t x) { return __fadd_rn(one_plus_m(x), -0.99999994039535522461f); }

__device__ __forceinline__ float ex2_approx(float x)
{
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
__device__ __forceinline__ float rcp_approx(float x)
{
    float y;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
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

// Packed fp32 pairs (sm_100a FFMA2 / FADD2 / FMUL2: two fp32 operations per issued instruction).
// In update_pair the two lanes of a pair are the two sites a thread has in flight.
__device__ __forceinline__ float2 add2(float2 a, float2 b) { return __fadd2_rn(a, b); }
__device__ __forceinline__ float2 mul2(float2 a, float2 b) { return __fmul2_rn(a, b); }
__device__ __forceinline__ float2 fma2(float2 a, float2 b, float2 c) { return __ffma2_rn(a, b, c); }
__device__ __forceinline__ float2 neg2(float2 a) { return make_float2(-a.x, -a.y); }
__device__ __forceinline__ float2 bc2(float a) { return make_float2(a, a); }

// sincos_small on a pair
__device__ __forceinline__ void sincos_small2(float2 x, float2& s, float2& c)
{
    const float2 x2 = mul2(x, x);
    float2 ps = fma2(x2, bc2(2.75573192e-6f), bc2(-1.98412698e-4f));
    ps = fma2(x2, ps, bc2(8.33333333e-3f));
    ps = fma2(x2, ps, bc2(-1.66666667e-1f));
    s = fma2(mul2(x, x2), ps, x);
    float2 pc = fma2(x2, bc2(-2.75573192e-7f), bc2(2.48015873e-5f));
    pc = fma2(x2, pc, bc2(-1.38888889e-3f));
    pc = fma2(x2, pc, bc2(4.16666667e-2f));
    pc = fma2(x2, pc, bc2(-0.5f));
    c = fma2(x2, pc, bc2(1.0f));
}

// the same for |x| <= SMALL_HD (proposal windows a >= q pi / (2 SMALL_HD)): sin to x^5 (truncation x^6/5040 < 2e-10
// relative), cos to x^4 (x^6/720 < 1.4e-9)
constexpr float SMALL_HD = 0.1f;
__device__ __forceinline__ void sincos_tiny2(float2 x, float2& s, float2& c)
{
    const float2 x2 = mul2(x, x);
    const float2 ps = fma2(x2, bc2(8.33333333e-3f), bc2(-1.66666667e-1f));
    s = fma2(mul2(x, x2), ps, x);
    const float2 pc = fma2(x2, bc2(4.16666667e-2f), bc2(-0.5f));
    c = fma2(x2, pc, bc2(1.0f));
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

__device__ __forceinline__ bool is_fixed(const uint32_t* __restrict__ bits, uint32_t n)
{
    return (bits[n >> 5] >> (n & 31)) & 1u;
}

// ---------------------------------------------------------------------------
// a1  min / max over the SAMPLE values, sample count, finiteness
// ---------------------------------------------------------------------------
__global__ void k_state_reset(Dev d)
{
    const int g = blockIdx.x * blockDim.x + threadIdx.x;
    if (g >= d.nv) return;
    GridState& s = d.states[g];
    s.t = 0; s.done = 0; s.cur = 0; s.hd_scale = 0.f; s.neg_log2e_over_T = 0.f;
    s.n_free[0] = s.n_free[1] = 0; s.max_tile_entries = 0;
    s.accepted = 0ull;
    s.zmin_enc = 0xFFFFFFFFu; s.zmax_enc = 0u;
    s.n_samples = 0; s.err_flags = 0; s.i = 0; s.realizations = 0;
    s.a = 1.0; s.k = -1.0; s.A_last = 0.0; s.e_last = 0.0; s.T = 0.0;
    s.zmin = 0.f; s.zmax = 0.f; s.e_query = 0.0; s.e_sum = 0.0; s.n_meas = 0; s.n_pairs = 0ull;
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
    const uint32_t n_end = (uint32_t)d.own_r1 * (uint32_t)d.cols;       // a slab's ghost rows belong to its neighbours
    for (uint32_t n = (uint32_t)d.own_r0 * (uint32_t)d.cols + blockIdx.x * blockDim.x + threadIdx.x; n < n_end; n += gridDim.x * blockDim.x) {
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

// unconditional grids (Alg. 2 step 4.2: every node free, no data): the angle is its own value
__global__ void k_state_unconditional(Dev d)
{
    const int g = blockIdx.x * blockDim.x + threadIdx.x;
    if (g >= d.batch) return;
    d.states[g].zmin = 0.0f; d.states[g].zmax = TWO_PI_F;
}

// ---------------------------------------------------------------------------
// a2  Eq. 1 at the sample sites, fixed-site bitmask, verbatim value copy,
// prediction-site count per checkerboard colour
// ---------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_transform(Dev d, const float* __restrict__ values,
                                                   const uint8_t* __restrict__ mask)
{
    const int g = blockIdx.y;
    const uint32_t n = blockIdx.x * blockDim.x + threadIdx.x;   // < 32 * words (grid sized so)
    const GridState& s = d.states[g];
    const bool in = n < d.N;
    bool fixed = false, own = false;
    uint32_t colour = 0;
    if (in) {
        const size_t o = (size_t)g * d.N + n;
        const float z = values ? values[o] : 0.0f;           // no inputs: an unconditional grid
        fixed = mask ? mask[o] != 0 : false;
        d.values[o] = z;
        d.phi[o] = fixed ? eq1(z, s.zmin, s.zmax) : 0.0f;
        const uint32_t r = n / d.cols;
        colour = (r + (n - r * d.cols)) & 1u;
        own = (int)r >= d.own_r0 && (int)r < d.own_r1;
    }
    const uint32_t b = __ballot_sync(0xFFFFFFFFu, fixed);
    const uint32_t f0 = __ballot_sync(0xFFFFFFFFu, in && own && !fixed && colour == 0);
    const uint32_t f1 = __ballot_sync(0xFFFFFFFFu, in && own && !fixed && colour == 1);
    // counts: per block in shared memory, then one global atomic per block and colour
    __shared__ uint32_t s_free[2];
    if (threadIdx.x < 2) s_free[threadIdx.x] = 0;
    __syncthreads();
    if ((threadIdx.x & 31) == 0 && (n >> 5) < d.words) {
        d.bits[(size_t)g * d.words + (n >> 5)] = b;
        if (f0) atomicAdd(&s_free[0], (uint32_t)__popc(f0));
        if (f1) atomicAdd(&s_free[1], (uint32_t)__popc(f1));
    }
    __syncthreads();
    if (threadIdx.x < 2 && s_free[threadIdx.x]) atomicAdd(&d.states[g].n_free[threadIdx.x], s_free[threadIdx.x]);
}

// ---------------------------------------------------------------------------
// a2  tile frames.  The grid is cut into TR x TC core tiles; a tile's frame is
// its core plus a halo of H sites on every side.  For each tile the free
// sites of the frame with ring < H (ring = Chebyshev distance outside the
// core, 0 inside) are listed per colour (checkerboard split),
// core first, then ring 1, 2, ..., so that the sites a half-sweep of a
// K-sweep pass still needs are a prefix of the list.  A half-warp of a
// 64-bit shared-memory access is served in one wavefront when its 16 lanes
// fall into 16 different eight-byte slots of a 128-byte line (slot = frame
// offset mod 16; the four neighbours shift every lane's slot alike).  The
// list is therefore built 16 entries at a time, each group taking sites of
// slots it does not hold yet, fullest slot first (k_tile_fill).
// ---------------------------------------------------------------------------
struct TileGeom { int r0, c0, TRc, TCc; };

__device__ __forceinline__ TileGeom tile_geom_xy(const Dev& d, int tx, int ty)
{
    TileGeom t;
    t.r0 = ty * d.TR; t.c0 = tx * d.TC;
    t.TRc = min(d.TR, d.rows - t.r0); t.TCc = min(d.TC, d.cols - t.c0);
    return t;
}
__device__ __forceinline__ TileGeom tile_geom(const Dev& d, int tile)
{
    const int ty = tile / d.ntx;
    return tile_geom_xy(d, tile - ty * d.ntx, ty);
}

// class of frame site (lr, lc): returns false if outside the grid, fixed, or on the outermost ring
__device__ __forceinline__ bool frame_site_class(const Dev& d, const uint32_t* __restrict__ bits, const TileGeom& t,
                                                 int lr, int lc, int& colour, int& ring)
{
    const int r = t.r0 - d.H + lr, col = t.c0 - d.H + lc;
    if (r < 0 || r >= d.rows || col < 0 || col >= d.cols) return false;
    if (is_fixed(bits, (uint32_t)r * d.cols + col)) return false;
    const int dr = max(max(d.H - lr, lr - (d.H + t.TRc - 1)), 0);
    const int dc = max(max(d.H - lc, lc - (d.H + t.TCc - 1)), 0);
    ring = max(dr, dc);
    colour = (r + col) & 1;
    return ring < d.H;
}

__global__ void __launch_bounds__(256) k_tile_count(Dev d)
{
    const int tile = blockIdx.x, g = blockIdx.y;
    __shared__ uint32_t hist[2][MAX_H];
    for (int i = threadIdx.x; i < 2 * MAX_H; i += blockDim.x) (&hist[0][0])[i] = 0;
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
        for (int k = 0; k < MAX_H; ++k) { run += hist[c][k]; m.cle[c][k] = run; }
    }
}

// one warp per grid: the largest entry count of a tile (two 16-aligned lists), which sizes the tile pass's
// shared memory and its entry-list copy
__global__ void k_tile_scan(Dev d)
{
    const int g = blockIdx.x;
    const uint32_t lane = threadIdx.x;
    const TileMeta* m = d.tile_meta + (size_t)g * d.ntiles;
    uint32_t mx = 0;
    for (int i = lane; i < d.ntiles; i += 32)
        mx = max(mx, (colour1_base(m[i].cle[0][MAX_H - 1]) + m[i].cle[1][MAX_H - 1] + 15u) & ~15u);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) mx = max(mx, __shfl_xor_sync(0xFFFFFFFFu, mx, o));
    if (lane == 0) d.states[g].max_tile_entries = mx;
}

// dynamic shared memory: FR * FC uint16 (the frame's free sites bucketed by colour, ring, slot)
__global__ void __launch_bounds__(256) k_tile_fill(Dev d)
{
    const int tile = blockIdx.x, g = blockIdx.y;
    extern __shared__ uint16_t bucketed[];
    __shared__ uint32_t cnt[2][MAX_H][16];       // free sites per (colour, ring, slot)
    __shared__ uint32_t start[2][MAX_H][16];     // bucket offsets in bucketed[]
    __shared__ uint32_t cursor[2][MAX_H][16];
    for (int i = threadIdx.x; i < 2 * MAX_H * 16; i += blockDim.x) { (&cnt[0][0][0])[i] = 0; (&cursor[0][0][0])[i] = 0; }
    __syncthreads();
    const TileGeom t = tile_geom(d, tile);
    const TileMeta& m = d.tile_meta[(size_t)g * d.ntiles + tile];
    const uint32_t* bits = d.bits + (size_t)g * d.words;
    uint16_t* out = d.entries + (size_t)g * d.entry_stride + (size_t)tile * d.tile_entries;
    for (int i = threadIdx.x; i < d.FR * d.FC; i += blockDim.x) {
        const int lr = i / d.FC, lc = i - lr * d.FC;
        int colour, ring;
        if (frame_site_class(d, bits, t, lr, lc, colour, ring)) atomicAdd(&cnt[colour][ring][i & 15], 1u);
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        uint32_t run = 0;
        for (int i = 0; i < 2 * MAX_H * 16; ++i) { (&start[0][0][0])[i] = run; run += (&cnt[0][0][0])[i]; }
    }
    __syncthreads();
    for (int i = threadIdx.x; i < d.FR * d.FC; i += blockDim.x) {
        const int lr = i / d.FC, lc = i - lr * d.FC;
        int colour, ring;
        if (frame_site_class(d, bits, t, lr, lc, colour, ring)) {
            const uint32_t b = i & 15;
            bucketed[start[colour][ring][b] + atomicAdd(&cursor[colour][ring][b], 1u)] = (uint16_t)i;
        }
    }
    __syncthreads();
    // warp c builds colour c's list: lane b < 16 owns slot b.  Every position takes the site of the slot
    // that occurs least in the current group of 16, fullest slot first.
    const int c = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (c >= 2) return;
    uint32_t pos = c ? colour1_base(m.cle[0][MAX_H - 1]) : 0u;
    uint32_t in_group = 0;                        // how often this lane's slot occurs in the current group
    for (int ring = 0; ring < d.H; ++ring) {
        uint32_t rem = lane < 16 ? cnt[c][ring][lane] : 0u;
        const uint32_t from = lane < 16 ? start[c][ring][lane] : 0u;
        uint32_t taken = 0;
        for (;;) {
            if ((pos & 15u) == 0u) in_group = 0;  // a new group starts
            const uint32_t key = rem ? ((15u - min(in_group, 15u)) << 24) | (min(rem, 0xFFFFFu) << 4) | (uint32_t)lane : 0u;
            const uint32_t best = __reduce_max_sync(0xFFFFFFFFu, key);
            if (best == 0u) break;
            if (lane == (int)(best & 15u)) {
                out[pos] = bucketed[from + taken];
                ++taken; --rem; ++in_group;
            }
            ++pos;
        }
    }
}

// The same lists in closed form, for grids that cannot fill the device.  Within a class (colour, ring) the list is built
// round by round: round k takes the k-th site of every slot that still has one, fullest slot first.  While all 16 slots
// have sites a round IS a conflict-free group of 16; the rounds after that hold what the fuller slots have left, which no
// order could serve in fewer wavefronts (a slot with m sites needs m of them).  The position of the k-th site of slot b
// follows from the class's 16 slot counts --
//   sum over the slots b' of min(count[b'], k)   (the sites of the rounds before k)
//   + the number of slots still in round k that come before b (larger count, or equal count and smaller b)
// -- so every site finds its place on its own: 10 x faster than k_tile_fill's walk (64 against 640 us at 4096^2), for 23 %
// more bank conflicts in the sweeps (the walk also fits a class's first entries to the previous class's last ones within
// a group of 16; measured on cfg4: 32.2 against 31.95 us per sweep).  Used where the passes wait on latency, not on
// shared-memory bandwidth, and the list walk was up to a quarter of a whole run.
__global__ void __launch_bounds__(256) k_tile_fill_rounds(Dev d)
{
    const int tile = blockIdx.x, g = blockIdx.y;
    __shared__ uint32_t cnt[2][MAX_H][16];       // free sites per (colour, ring, slot)
    __shared__ uint32_t cursor[2][MAX_H][16];
    __shared__ uint32_t base[2][MAX_H];          // list position of the class's first entry
    for (int i = threadIdx.x; i < 2 * MAX_H * 16; i += blockDim.x) { (&cnt[0][0][0])[i] = 0; (&cursor[0][0][0])[i] = 0; }
    __syncthreads();
    const TileGeom t = tile_geom(d, tile);
    const TileMeta& m = d.tile_meta[(size_t)g * d.ntiles + tile];
    const uint32_t* bits = d.bits + (size_t)g * d.words;
    uint16_t* out = d.entries + (size_t)g * d.entry_stride + (size_t)tile * d.tile_entries;
    for (int i = threadIdx.x; i < d.FR * d.FC; i += blockDim.x) {
        const int lr = i / d.FC, lc = i - lr * d.FC;
        int colour, ring;
        if (frame_site_class(d, bits, t, lr, lc, colour, ring)) atomicAdd(&cnt[colour][ring][i & 15], 1u);
    }
    if (threadIdx.x < 2 * MAX_H) {
        const int c = threadIdx.x / MAX_H, r = threadIdx.x % MAX_H;
        base[c][r] = (c ? colour1_base(m.cle[0][MAX_H - 1]) : 0u) + (r ? m.cle[c][r - 1] : 0u);
    }
    __syncthreads();
    for (int i = threadIdx.x; i < d.FR * d.FC; i += blockDim.x) {
        const int lr = i / d.FC, lc = i - lr * d.FC;
        int colour, ring;
        if (!frame_site_class(d, bits, t, lr, lc, colour, ring)) continue;
        const uint32_t b = i & 15;
        const uint32_t k = atomicAdd(&cursor[colour][ring][b], 1u), mine = cnt[colour][ring][b];
        uint32_t pos = base[colour][ring];
#pragma unroll
        for (uint32_t o = 0; o < 16; ++o) {
            const uint32_t n = cnt[colour][ring][o];
            pos += min(n, k) + ((n > k && (n > mine || (n == mine && o < b))) ? 1u : 0u);
        }
        out[pos] = (uint16_t)i;
    }
}

// ---------------------------------------------------------------------------
// a2  initial state (Alg. 2 step 2.2, L176): phi ~ U(0, 2 pi) at prediction
// sites from the INIT stream; every site's unit vector (cos q phi, sin q phi)
// into BOTH vector buffers (sample sites are never written again).
// ---------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_init_state(Dev d, int ordered)
{
    const int g = blockIdx.y;
    const uint32_t n = blockIdx.x * blockDim.x + threadIdx.x;
    if (n >= d.N) return;
    const size_t o = (size_t)g * d.N + n;
    float p;
    if (is_fixed(d.bits + (size_t)g * d.words, n)) p = d.phi[o];
    else {
        if (ordered) p = 3.14159274101257324f;          // unconditional chains start from phi = pi (reading R23)
        else {
            const uint32_t ng = n + d.site_off;             // the site's index in the whole grid (a slab's rows start at slab_row0)
            const uint4 x = philox4x32_10(ng >> 2, 0u, 0u, (uint32_t)g, d.rk0, d.rk1);
            const uint32_t w = (ng & 3u) == 0 ? x.x : (ng & 3u) == 1 ? x.y : (ng & 3u) == 2 ? x.z : x.w;
            p = __fmul_rn(TWO_PI_F, u01(w));
        }
        d.phi[o] = p;
    }
    const uint32_t r = n / d.cols, col = n - r * d.cols;
    float sn, cs;
    sincosf(__fmul_rn(d.q, p), &sn, &cs);
    const size_t at = (size_t)r * d.pitch + col;
    vec_grid(d, g, 0)[at] = make_float2(cs, sn);
    vec_grid(d, g, 1)[at] = make_float2(cs, sn);
}

// ---------------------------------------------------------------------------
// a3  UPDATE of one prediction site (Alg. 1) in vector form.
// v = (cos q phi, sin q phi); (hx, hy) = (C, S) = sum over the neighbours.
// w0, w1: the two random words of this site and sweep (R13).
// ---------------------------------------------------------------------------
template <bool QHALF, int ORMODE>
__device__ __forceinline__ float2 update_site(float2 v, float2 n_up, float2 n_dn, float2 n_lf, float2 n_rt,
                                              uint32_t w0, uint32_t w1, float hd_scale, float hd_c1, float nlT,
                                              float bc, float bs, bool& accepted)
{
    const float hx = (n_up.x + n_dn.x) + (n_lf.x + n_rt.x), hy = (n_up.y + n_dn.y) + (n_lf.y + n_rt.y);
    float px = v.x, py = v.y;
    // Alg. 1 line 1: over-relaxation.  Reflect v about h: q phi' = 2 Theta - q phi keeps h.v,
    // i.e. the local energy (L156, L265; R2).  Out of [0, 2 pi]: keep the spin.
    if (ORMODE == 0) {
        const float R2 = fmaf(hx, hx, hy * hy);
        const float dot = fmaf(px, hx, py * hy);
        const float k = (dot + dot) * rcp_approx(R2);                    // 0 * inf -> NaN -> kept below
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
    // lines 2-3: phi'' = phi' + 2 pi (u - 1/2)/a (mod 2 pi): rotate by d = q delta = 2 hd, with
    // hd = (u - 1/2) hd_scale = (g + 2^-24) hd_scale, g = 1.m - 1.5 exact, hd_c1 = 2^-24 hd_scale
    const float hd = fmaf(__fadd_rn(one_plus_m(w0), -1.5f), hd_scale, hd_c1);
    float sh, ch;
    sincos_small(hd, sh, ch);
    const float sh2 = sh + sh;
    const float sd = sh2 * ch, omc = sh2 * sh;                           // sin d, 1 - cos d
    float rx = fmaf(-sd, py, fmaf(-omc, px, px));
    float ry = fmaf(sd, px, fmaf(-omc, py, py));
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
    accepted = dH <= 0.0f || ex2_approx(dH * nlT) > u01(w1);
    return make_float2(accepted ? rx : px, accepted ? ry : py);
}

// The same UPDATE for the two sites A and B a thread has in flight, with the fp32 arithmetic of both packed
// into f32x2 instructions (lane x = site A, lane y = site B).  Identities used on top of update_site:
// the reflection keeps h.v, so h.v' = h.v, and turns h x v into -(h x v); both are taken from the stored v,
// which is what the oracle's exact arithmetic does (it does not round v' before the Metropolis step).
// exp(-dH/T) > r already accepts every dH <= 0 because r < 1.
template <bool QHALF, int ORMODE, bool SMALLD>
__device__ __forceinline__ void update_pair(float2& vA, float2 upA, float2 dnA, float2 lfA, float2 rtA,
                                            float2& vB, float2 upB, float2 dnB, float2 lfB, float2 rtB,
                                            uint32_t wA0, uint32_t wA1, uint32_t wB0, uint32_t wB1,
                                            float hd_scale, float hd_c1, float nlT, float bc, float bs, bool renorm,
                                            bool& accA, bool& accB)
{
    if (ORMODE == 1) {      // Eq. 6 as printed: comparison mode, not packed
        vA = update_site<QHALF, ORMODE>(vA, upA, dnA, lfA, rtA, wA0, wA1, hd_scale, hd_c1, nlT, bc, bs, accA);
        vB = update_site<QHALF, ORMODE>(vB, upB, dnB, lfB, rtB, wB0, wB1, hd_scale, hd_c1, nlT, bc, bs, accB);
        if (renorm) {
            const float sA = fmaf(-0.5f, fmaf(vA.x, vA.x, vA.y * vA.y), 1.5f), sB = fmaf(-0.5f, fmaf(vB.x, vB.x, vB.y * vB.y), 1.5f);
            vA = make_float2(vA.x * sA, vA.y * sA); vB = make_float2(vB.x * sB, vB.y * sB);
        }
        return;
    }
    // Two packings are used so that no register moves are needed: (x, y) of ONE site for what is linear in
    // the vectors (the registers a 64-bit shared load fills), and (site A, site B) for the scalar chain.
    // (C, S) = h per site
    const float2 hA = add2(add2(upA, dnA), add2(lfA, rtA));
    const float2 hB = add2(add2(upB, dnB), add2(lfB, rtB));
    const float2 hvA = mul2(hA, vA), hvB = mul2(hB, vB);
    const float2 dot = make_float2(hvA.x + hvA.y, hvB.x + hvB.y);            // h . v  (= h . v')
    float2 crs = make_float2(fmaf(hA.x, vA.y, -hA.y * vA.x), fmaf(hB.x, vB.y, -hB.y * vB.x));   // h x v
    float2 pA = vA, pB = vB;
    if (ORMODE == 0) {
        // Alg. 1 line 1: over-relaxation, v' = 2 (h.v)/(h.h) h - v; out of [0, 2 pi]: keep the spin (R2, R17);
        // h x v' = -(h x v)
        const float2 hhA = mul2(hA, hA), hhB = mul2(hB, hB);
        const float2 R2 = make_float2(hhA.x + hhA.y, hhB.x + hhB.y);
        const float2 rinv = make_float2(rcp_approx(R2.x), rcp_approx(R2.y));      // 0 * inf -> NaN -> kept
        const float2 t = mul2(dot, rinv);
        const float2 k = add2(t, t);
        const float2 fA = fma2(hA, bc2(k.x), neg2(vA)), fB = fma2(hB, bc2(k.y), neg2(vB));
        bool inA = fA.y >= 0.0f && hA.y >= 0.0f, inB = fB.y >= 0.0f && hB.y >= 0.0f;
        if (!QHALF) {
            inA = inA && fmaf(fA.x, bs, -fA.y * bc) >= 0.0f;
            inB = inB && fmaf(fB.x, bs, -fB.y * bc) >= 0.0f;
        }
        pA = make_float2(inA ? fA.x : vA.x, inA ? fA.y : vA.y);
        pB = make_float2(inB ? fB.x : vB.x, inB ? fB.y : vB.y);
        crs = make_float2(inA ? -crs.x : crs.x, inB ? -crs.y : crs.y);
    }
    // lines 2-3: rotate v' by d = q delta = 2 hd, hd = (u - 1/2) hd_scale = (g + 2^-24) hd_scale,
    // g = 1.m - 1.5 exact, hd_c1 = 2^-24 hd_scale
    const float2 hd = fma2(add2(make_float2(one_plus_m(wA0), one_plus_m(wB0)), bc2(-1.5f)), bc2(hd_scale), bc2(hd_c1));
    float2 sh, ch;
    if (SMALLD) sincos_tiny2(hd, sh, ch); else sincos_small2(hd, sh, ch);
    const float2 sh2 = add2(sh, sh);
    const float2 sd = mul2(sh2, ch), omc = mul2(sh2, sh);       // sin d, 1 - cos d
    const float2 tA = fma2(pA, bc2(-omc.x), pA), tB = fma2(pB, bc2(-omc.y), pB);
    float rxA = fmaf(-sd.x, pA.y, tA.x), ryA = fmaf(sd.x, pA.x, tA.y);
    float rxB = fmaf(-sd.y, pB.y, tB.x), ryB = fmaf(sd.y, pB.x, tB.y);
    // line 4: dH = -h.(v'' - v') = (1 - cos d)(h.v') + sin d (h x v')
    float2 dH = fma2(omc, dot, mul2(sd, crs));
    if (QHALF) {
        // q = 1/2: q phi in [0, pi]; leaving it <=> sin < 0; phi -/+ 2 pi <=> v -> -v
        if (ryA < 0.0f) { rxA = -rxA; ryA = -ryA; dH.x = fmaf(2.0f, dot.x, -dH.x); }
        if (ryB < 0.0f) { rxB = -rxB; ryB = -ryB; dH.y = fmaf(2.0f, dot.y, -dH.y); }
    } else {
        const bool underA = hd.x < 0.0f && ryA < 0.0f, overA = hd.x > 0.0f && !(ryA >= 0.0f && fmaf(rxA, bs, -ryA * bc) >= 0.0f);
        const bool underB = hd.y < 0.0f && ryB < 0.0f, overB = hd.y > 0.0f && !(ryB >= 0.0f && fmaf(rxB, bs, -ryB * bc) >= 0.0f);
        if (underA || overA) {
            const float s2 = underA ? bs : -bs;
            const float wx = fmaf(rxA, bc, -ryA * s2), wy = fmaf(rxA, s2, ryA * bc);
            rxA = wx; ryA = wy;
            dH.x = dot.x - fmaf(hA.x, wx, hA.y * wy);
        }
        if (underB || overB) {
            const float s2 = underB ? bs : -bs;
            const float wx = fmaf(rxB, bc, -ryB * s2), wy = fmaf(rxB, s2, ryB * bc);
            rxB = wx; ryB = wy;
            dH.y = dot.y - fmaf(hB.x, wx, hB.y * wy);
        }
    }
    // lines 5-6: AP = min{1, exp(-dH/T)}; accept phi'' if AP > r else keep phi'
    const float2 arg = mul2(dH, bc2(nlT));
    const float2 r = add2(make_float2(one_plus_m(wA1), one_plus_m(wB1)), bc2(-0.99999994039535522461f));
    accA = ex2_approx(arg.x) > r.x;
    accB = ex2_approx(arg.y) > r.y;
    vA = make_float2(accA ? rxA : pA.x, accA ? ryA : pA.y);
    vB = make_float2(accB ? rxB : pB.x, accB ? ryB : pB.y);
    if (renorm) {           // first-order Newton step of 1/|v|
        const float2 nA = mul2(vA, vA), nB = mul2(vB, vB);
        vA = mul2(vA, bc2(fmaf(-0.5f, nA.x + nA.y, 1.5f)));
        vB = mul2(vB, bc2(fmaf(-0.5f, nB.x + nB.y, 1.5f)));
    }
}

// ---------------------------------------------------------------------------
// a6  equilibration controller: Alg. 2 steps 5.2-5.5 for
// one grid, by ONE thread, after the sweep (5.1) whose accepted proposals sit in
// GridState::accepted and whose energy is H.  Commits the sweep: t += 1 and the
// vector buffers swap roles.  Called by k_controller (one block per grid after a
// K = 1 tile pass) and, for a grid that is a single tile, from inside the tile pass.
// ---------------------------------------------------------------------------
// s: the grid's state, in global memory or a copy of it (the tile pass keeps one in shared memory while it loops)
__device__ __forceinline__ void controller_step(const Dev& d, GridState& s, double H, double P_total = 0.0)
{
    const uint32_t i = s.i;
    const double P = P_total > 0.0 ? P_total : (double)s.n_free[0] + (double)s.n_free[1];
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
    // unconditional chains burn in for exactly equil_cap sweeps: from their ordered start the energy rises, so the
    // slope criterion would stop them at its first check (reading R23)
    const bool go_on = d.burn_in_only ? i + 1u < d.equil_cap : (k < 0.0 && i + 1u < d.equil_cap);
    if (!go_on) s.done = 1u;
}

// ---- TMA / mbarrier PTX (sm_100a) -------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity)
{
    uint32_t done;
    do {
        asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                     : "=r"(done) : "r"(smem_u32(bar)), "r"(parity) : "memory");
    } while (!done);
}
// frame box (FC x FR x 1 eight-byte elements) of the vector buffer; out-of-grid elements arrive as zeros
__device__ __forceinline__ void tma_load_frame(void* dst, const CUtensorMap* map, int c, int r, int g, uint64_t* bar)
{
    asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];"
                 ::"r"(smem_u32(dst)), "l"((uint64_t)map), "r"(c), "r"(r), "r"(g), "r"(smem_u32(bar)) : "memory");
}
// L2 prefetch of a frame box / of a byte range (no shared-memory destination, no completion to wait for)
__device__ __forceinline__ void tma_prefetch_frame(const CUtensorMap* map, int c, int r, int g)
{
    asm volatile("cp.async.bulk.prefetch.tensor.3d.L2.global.tile [%0, {%1, %2, %3}];"
                 ::"l"((uint64_t)map), "r"(c), "r"(r), "r"(g) : "memory");
}
__device__ __forceinline__ void bulk_prefetch(const void* src, uint32_t bytes)
{
    asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"((uint64_t)src), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_load(void* dst, const void* src, uint32_t bytes, uint64_t* bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(dst)), "l"((uint64_t)src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void bulk_store(void* dst, const void* src, uint32_t bytes)
{
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;"
                 ::"l"((uint64_t)dst), "r"(smem_u32(src)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_commit_wait_read()
{
    asm volatile("cp.async.bulk.commit_group;" ::: "memory");
    asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
}
// programmatic dependent launch (no-ops in a kernel launched without the attribute)
__device__ __forceinline__ void griddep_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
__device__ __forceinline__ void griddep_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void fence_proxy_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

// ---------------------------------------------------------------------------
// a3/a4  the hot kernel: K whole sweeps (colour 0 then colour 1, L261-265) of
// one tile, on a copy of its frame in shared memory (temporal blocking).
// The frame arrives by one TMA tensor load (out-of-grid sites as zero vectors
// = open boundary) together with the tile's entry list; the
// tile's core leaves by one bulk copy per row into the OTHER vector buffer, so
// tiles of one launch never see each other's writes.  Sites of the halo are
// updated redundantly; they reproduce the neighbouring tiles' results bit for
// bit because the random numbers are keyed by (site, sweep).  After half-sweep
// number hs (0-based) the frame is valid up to ring 2K-1-hs, so each
// half-sweep only updates the prefix of the entry list with ring <= 2K-1-hs.
// Every thread keeps two sites in flight and their arithmetic shares f32x2
// instructions (update_pair).  Optionally fused at the end:
//   PASS_ENERGY      a5: - sum over the core's colour-1 sites of v.h (each bond once)   [FUSED only]
//   PASS_COUNT       a5: accepted proposals of the core sites                          [FUSED only]
//   PASS_ACCUMULATE  a7: acc += phi at the core's prediction sites (and the squared deviations for L212)
// ---------------------------------------------------------------------------
// a5 inside a tile pass: this warp's share of sum over the core's colour-1 sites (fixed ones too) of v . h, rows dealt
// over the warps, float per row, double over the rows, then the warp's shuffle tree: a fixed order
__device__ __forceinline__ double core_energy_warp(const Dev& d, const float2* S, const TileGeom& tg, int H, int FC, int warp, int lane, int NW)
{
    double sum = 0.0;
    for (int lr = H + warp; lr < H + tg.TRc; lr += NW) {
        const int r = tg.r0 - H + lr;
        if (r < d.own_r0 || r >= d.own_r1) continue;         // a slab's ghost rows are counted by the slab that owns them
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
    return sum;
}

// what one half-sweep of a tile pass needs to know (tabulated per CTA, see k_tilepass)
struct __align__(16) HalfSweep { uint32_t n, cbase, c1, flags; };   // entries to walk, list offset, Philox counter word 1, HS_*
enum : uint32_t { HS_ODD = 1u, HS_FRESH = 2u, HS_STASH = 4u, HS_RENORM = 8u, HS_ACC = 16u };   // bits 8: colour, 16..: realization offset
constexpr int HS_CHUNK = 16;

// how a half-sweep gets its random words: the stored second pair, a Philox draw of an even sweep whose second pair is
// stored (the usual drawing sweep), or a draw in general (odd sweep at the start of a pass, no room for stored words)
enum { DRAW_STORED = 0, DRAW_EVEN_STORE = 1, DRAW_ANY = 2 };
template <int M> struct DrawTag { static constexpr int value = M; };

// EQUIL (a grid that is ONE tile, with FUSED): Alg. 2 step 5 runs inside the pass -- after every sweep the energy and
// the accepted count are reduced in the CTA, thread 0 takes steps 5.2-5.5 (controller_step) and the CTA goes on with the
// new proposal width or stops; K is then the most sweeps this launch may do.  Bit for bit the sweeps of the K = 1
// passes with k_controller between them, without 2 launches per sweep.
// MINB: CTAs per SM the registers are budgeted for: 3 for the K-sweep passes (their shared memory allows no more), 4 for
// single-sweep passes (row halo 2, no stored random words: 49 KB), whose length is mostly a CTA's own latency
template <bool QHALF, int ORMODE, bool FUSED, int FCT, bool SMALLD, bool EQUIL = false, int MINB = 3>
__global__ void __launch_bounds__(TILE_THREADS, MINB)
k_tilepass(const __grid_constant__ CUtensorMap map0, const __grid_constant__ CUtensorMap map1, const Dev d,
           uint32_t K, uint32_t t_off, uint32_t src_sel, uint32_t flags, uint32_t pf_dist, uint32_t real_no, uint32_t row_halo,
           uint32_t g_first, uint32_t acc_every)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    __shared__ __align__(8) uint64_t s_bar[2];       // [0] frame, [1] entry list
    __shared__ uint32_t s_cle[2][MAX_H];
    __shared__ HalfSweep s_hs[HS_CHUNK];
    __shared__ uint32_t s_accepted;
    __shared__ double s_red[TILE_THREADS / 32];

    constexpr int NT = TILE_THREADS, NW = TILE_THREADS / 32;
    static_assert(TILE_THREADS >= 96 + 2 * MAX_H && TILE_THREADS >= HS_CHUNK, "the prologue gives warps 0-3 their own jobs");
    // grid = (tiles across, tiles down, states): the tile's place without a division at the head of every CTA's life
    const int tile = (int)(blockIdx.y * gridDim.x + blockIdx.x), g = (int)(blockIdx.z + g_first);   // g: state (grid and chain), gd: the grid whose data it shares
    const int gd = g < d.batch ? g : g % d.batch;
    const GridState& st = d.states[g];
    // Programmatic dependent launch: the next kernel of the stream may start its CTAs while the last of this
    // one still run.  What a tile pass does before its own griddep_wait() touches only data no kernel of a run
    // writes (tile lists) and its own shared memory.
    griddep_launch_dependents();

    // frame pitch: a compile-time constant for the standard tile shape (neighbour offsets become immediates)
    const int H = d.H, FC = FCT ? FCT : d.FC;
    const uint32_t fc_inv = FCT ? (uint32_t)(((1u << 24) + (uint32_t)(FCT ? FCT : 1) - 1u) / (uint32_t)(FCT ? FCT : 1)) : d.fc_inv;
    // A pass of K sweeps needs 2K rings of halo.  The frame that is loaded keeps the full pitch FC (entry offsets are
    // row * FC + col of the full frame) but only row_halo = min(H, 2K) halo rows above and below the core: the maps'
    // box has TR + 2 row_halo rows.  S points where row 0 of the FULL frame would be, so that the offsets stay valid;
    // rows above S_load are never touched (an entry of ring <= 2K - 1 has its upper neighbour in ring <= 2K).
    const int HR = (int)row_halo, FRK = d.TR + 2 * HR;
    float2*   S_load = reinterpret_cast<float2*>(smem_raw);
    uint32_t  s_shift = (uint32_t)((H - HR) * FC) * (uint32_t)sizeof(float2);
    asm volatile("" : "+r"(s_shift));    // opaque, so that the shifted base is formed once (else the shift is redone per site)
    float2*   S  = reinterpret_cast<float2*>(smem_raw - s_shift);
    uint2*    SP = reinterpret_cast<uint2*>(S_load + FRK * FC);
    uint16_t* E  = reinterpret_cast<uint16_t*>(SP + (d.use_spare ? d.max_entries : 0u));

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const TileGeom tg = tile_geom_xy(d, (int)blockIdx.x, (int)blockIdx.y);
    const TileMeta& meta = d.tile_meta[(size_t)gd * d.ntiles + tile];

    // three warps start the tile: warp 1 the entry list (needs the tile's counts from global memory first), and,
    // once the previous kernel's results are visible, warp 0 the frame and warp 2 the L2 prefetch
    if (tid == 0) { mbar_init(&s_bar[0], 1); s_accepted = 0; }
    else if (tid == 32) {
        // the entry list: always the size of the largest tile's (the rest of this tile's room is never indexed),
        // from a place that depends on the tile number only -- nothing has to be read first
        mbar_init(&s_bar[1], 1);
        const uint32_t entry_bytes = d.max_entries * (uint32_t)sizeof(uint16_t);
        mbar_expect_tx(&s_bar[1], entry_bytes);
        if (entry_bytes) bulk_load(E, d.entries + (size_t)gd * d.entry_stride + (size_t)tile * d.tile_entries, entry_bytes, &s_bar[1]);
    }
    if (tid >= 96 && tid < 96 + 2 * MAX_H) (&s_cle[0][0])[tid - 96] = (&meta.cle[0][0])[tid - 96];

    griddep_wait();         // from here on: the vector buffers and the grids' states as the previous kernels left them
    if (FUSED && (flags & PASS_CHECK_DONE) && st.done) {        // this grid's equilibration has stopped
        __syncthreads();
        mbar_wait(&s_bar[1], 0);                                 // no copy into this CTA's shared memory is left in flight
        return;
    }
    // src_sel 0 / 1: the source buffer is known to the host (every grid alike); 2: per grid, from its state
    const uint32_t src_buf = src_sel < 2u ? src_sel : st.cur;
    float2* dst = vec_grid(d, g, src_buf ^ 1u);
    if (tid == 0) {
        mbar_expect_tx(&s_bar[0], (uint32_t)(FRK * FC * sizeof(float2)));
        tma_load_frame(S_load, src_buf ? &map1 : &map0, tg.c0 - H, tg.r0 - HR, g, &s_bar[0]);
    }
    // warp 2 pulls what the tile that will run in this CTA slot next needs towards L2: its frame and its entry list
    if (tid == 64 && pf_dist && tile + (int)pf_dist < d.ntiles) {
        const TileGeom tn = tile_geom(d, tile + (int)pf_dist);
        tma_prefetch_frame(src_buf ? &map1 : &map0, tn.c0 - H, tn.r0 - HR, g);
        if (d.max_entries)
            bulk_prefetch(d.entries + (size_t)gd * d.entry_stride + (size_t)(tile + pf_dist) * d.tile_entries,
                          d.max_entries * (uint32_t)sizeof(uint16_t));
    }
    if (tid == 65 && (flags & PASS_ACCUMULATE)) {       // the tile's accumulators towards L2 while the sweeps run
        const size_t at = ((size_t)g * d.ntiles + tile) * d.acc_stride;
        const uint32_t bytes = ((uint32_t)(tg.TRc * tg.TCc) * 4u + 15u) & ~15u;      // never more than the tile can hold
        bulk_prefetch(d.acc + at, bytes);
        bulk_prefetch(d.m2 + at, bytes);
    }
    float hs = st.hd_scale, hc1 = hs * 5.9604644775390625e-08f;
    const float nlT = st.neg_log2e_over_T;
    __shared__ float s_ctrl[2];            // EQUIL: the controller's verdict for the CTA: new hd_scale, stop flag
    bool finished = false;
    GridState* s_state = nullptr;          // EQUIL: the grid's state while the CTA loops (written back at the end)
    if constexpr (EQUIL) {
        __shared__ GridState s_state_copy;
        s_state = &s_state_copy;
        for (uint32_t w = tid; w < sizeof(GridState) / 4; w += NT)
            reinterpret_cast<uint32_t*>(s_state)[w] = reinterpret_cast<const uint32_t*>(&d.states[g])[w];
    }
    const uint32_t t0 = st.t + t_off;
    const int nbase = (tg.r0 - H) * d.cols + (tg.c0 - H) + (int)d.site_off, ncorr = d.cols - FC;
    const bool count = FUSED && (flags & PASS_COUNT);
    // frame offsets [own_lo, own_lo + own_span) are the rows this context owns (all of them unless it is a slab)
    const uint32_t own_lo = (uint32_t)max(d.own_r0 - (tg.r0 - H), 0) * (uint32_t)FC;
    const uint32_t own_span = (uint32_t)max(min(d.own_r1 - (tg.r0 - H), d.FR) * FC - (int)own_lo, 0);
    const bool use_spare = d.use_spare;
    uint32_t n_accepted = 0;
    __syncthreads();
    // What a half-sweep needs to know is tabulated by one warp for 16 half-sweeps at a time (HalfSweep), so that the other
    // warps do not redo it; the first 16 while the frame is still on its way.
    auto fill_table = [&](uint32_t j0) {
        if (tid < HS_CHUNK && j0 + tid < 2u * K) {
            const uint32_t j = j0 + tid, s = j >> 1, c = j & 1u, t = t0 + s;
            const bool odd = t & 1u;
            const bool fresh = !odd || s == 0 || !use_spare;            // draw a new Philox block for (site, t >> 1)
            const bool stash = use_spare && !odd && s + 1 < K;          // keep words 2,3 for sweep t + 1
            // |v| = 1 against rounding drift, every fourth sweep BY THE GLOBAL SWEEP INDEX: which sweeps renormalise does
            // not depend on how they are grouped into passes, so neither does any bit of the state (a tile's halo
            // sites and its neighbour's core sites must renormalise alike anyway)
            const bool renorm = (t & 3u) == 3u;
            // step 6.3 inside the pass: after every acc_every-th sweep the core is accumulated (several realizations of
            // fewer than K sweeps per launch)
            const bool acc = (flags & PASS_ACCUMULATE) && c == 1u && (s + 1u) % acc_every == 0u;
            const uint32_t R = 2u * K - 1u - j;                          // rings still needed: 0 .. R
            HalfSweep h;
            h.n = s_cle[c][R < (uint32_t)MAX_H ? R : (uint32_t)MAX_H - 1u];
            h.cbase = c ? colour1_base(s_cle[0][MAX_H - 1]) : 0u;
            h.c1 = t >> 1;
            h.flags = (odd ? HS_ODD : 0u) | (fresh ? HS_FRESH : 0u) | (stash ? HS_STASH : 0u) | (renorm ? HS_RENORM : 0u) |
                      (acc ? HS_ACC : 0u) | (c << 8) | (acc ? ((s + 1u) / acc_every - 1u) << 16 : 0u);
            s_hs[tid] = h;
        }
    };
    fill_table(0u);
    mbar_wait(&s_bar[1], 0);
    mbar_wait(&s_bar[0], 0);

    auto accumulate_core = [&](uint32_t k) {
        // a7 (Alg. 2 step 6, L207-211): acc += phi at the core's prediction sites; and for the spread of the
        // realizations (L212) the sum of squared deviations, updated from the running mean so that nothing cancels:
        // m2 += (phi - mean_{k-1}) (phi - mean_k), k = number of this realization.
        // The accumulators are kept per tile in the order of the tile's core entries, so that a pass touches only
        // prediction sites' words, consecutive lanes consecutive words (and the tile's range was sent for at the start).
        float* acc = d.acc + ((size_t)g * d.ntiles + tile) * d.acc_stride;
        float* m2 = d.m2 + ((size_t)g * d.ntiles + tile) * d.acc_stride;
        const float inv_km1 = k > 1u ? 1.0f / (float)(k - 1u) : 0.0f, inv_k = 1.0f / (float)k;
        const uint32_t n0 = s_cle[0][0], a1 = colour1_base(n0), n_acc = a1 + s_cle[1][0], e1 = colour1_base(s_cle[0][MAX_H - 1]);
        // position i of the tile's accumulators: colour 0's core entry i (i < n0), colour 1's core entry i - a1 (i >= a1)
#pragma unroll 1
        for (uint32_t i0 = tid; i0 < n_acc; i0 += 4u * NT) {
            float a_[4], m_[4];
            bool on[4];
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const uint32_t i = i0 + (uint32_t)u * NT;
                on[u] = i < n_acc && (i < n0 || i >= a1);
                if (on[u]) { a_[u] = acc[i]; m_[u] = k > 1u ? m2[i] : 0.0f; }
            }
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                if (!on[u]) continue;
                const uint32_t i = i0 + (uint32_t)u * NT;
                const uint32_t off = E[i < n0 ? i : e1 + (i - a1)];
                MPR_CHECK(i < d.acc_stride && (i < n0 ? i : e1 + (i - a1)) < d.max_entries);
                MPR_CHECK(off >= (uint32_t)(H * FC + H) && off < (uint32_t)((H + tg.TRc) * FC));      // a core site
                const float phi = angle_of(S[off], d.inv_q), before = a_[u], after = before + phi;
                acc[i] = after;
                if (k > 1u) m2[i] = m_[u] + (phi - before * inv_km1) * (phi - after * inv_k);
            }
        }
    };

    // half-sweep j = 2 s + c: colour c of sweep s (Alg. 1: colour 0, then colour 1).  What a half-sweep needs to
    // know is tabulated by one warp for 16 half-sweeps at a time (HalfSweep), so that the other warps do not redo it.
#pragma unroll 1
    for (uint32_t j0 = 0; j0 < 2u * K && !(EQUIL && finished); j0 += HS_CHUNK) {
        if (j0) fill_table(j0);
        __syncthreads();
        const uint32_t j_end = min(2u * K - j0, (uint32_t)HS_CHUNK);
#pragma unroll 1
      for (uint32_t jj = 0; jj < j_end && !(EQUIL && finished); ++jj) {
        const HalfSweep h = s_hs[jj];
        const bool odd = h.flags & HS_ODD, fresh = h.flags & HS_FRESH, stash = h.flags & HS_STASH, renorm = h.flags & HS_RENORM;
        const uint32_t n = h.n, tc1 = h.c1;
        const uint32_t n_core = FUSED ? s_cle[(h.flags >> 8) & 1u][0] : 0u;
        const uint16_t* Ec = E + h.cbase;
        uint2* SPc = SP + h.cbase;

        // the sites eA and eB of this colour's list (eB == eA: no second site, its result is dropped).
        // The draw mode is a compile-time tag so that the Philox rounds and the update arithmetic of a drawing
        // sweep sit in one basic block (independent instruction streams for the scheduler to interleave).
        auto update_two = [&](auto draw_tag, uint32_t eA, uint32_t eB) {
            constexpr int DRAW = decltype(draw_tag)::value;
            MPR_CHECK(h.cbase + eA < d.max_entries && h.cbase + eB < d.max_entries);
            const uint32_t offA = Ec[eA], offB = Ec[eB];
            // the site and its four neighbours lie in the rows that were loaded, and never in the frame's first or last column
            MPR_CHECK(offA >= (uint32_t)((H - HR + 1) * FC + 1) && offA + (uint32_t)FC + 1u < (uint32_t)((H - HR + FRK) * FC));
            MPR_CHECK(offB >= (uint32_t)((H - HR + 1) * FC + 1) && offB + (uint32_t)FC + 1u < (uint32_t)((H - HR + FRK) * FC));
            float2 vA = S[offA], vB = S[offB];
            const float2 upA = S[offA - FC], dnA = S[offA + FC], lfA = S[offA - 1], rtA = S[offA + 1];
            const float2 upB = S[offB - FC], dnB = S[offB + FC], lfB = S[offB - 1], rtB = S[offB + 1];
            uint32_t wA0, wA1, wB0, wB1;
            if (DRAW != DRAW_STORED) {
                const uint32_t nA = (uint32_t)(nbase + (int)offA + (int)((offA * fc_inv) >> 24) * ncorr);
                const uint32_t nB = (uint32_t)(nbase + (int)offB + (int)((offB * fc_inv) >> 24) * ncorr);
                const uint4 xA = philox4x32_10(nA, tc1, 2u, (uint32_t)g, d.rk0, d.rk1);
                const uint4 xB = philox4x32_10(nB, tc1, 2u, (uint32_t)g, d.rk0, d.rk1);
                if (DRAW == DRAW_EVEN_STORE) {
                    wA0 = xA.x; wA1 = xA.y; wB0 = xB.x; wB1 = xB.y;
                    SPc[eA] = make_uint2(xA.z, xA.w); SPc[eB] = make_uint2(xB.z, xB.w);
                } else {
                    wA0 = odd ? xA.z : xA.x; wA1 = odd ? xA.w : xA.y;
                    wB0 = odd ? xB.z : xB.x; wB1 = odd ? xB.w : xB.y;
                    if (stash) { SPc[eA] = make_uint2(xA.z, xA.w); SPc[eB] = make_uint2(xB.z, xB.w); }
                }
            } else {
                const uint2 sA = SPc[eA], sB = SPc[eB];
                wA0 = sA.x; wA1 = sA.y; wB0 = sB.x; wB1 = sB.y;
            }
            bool accA, accB;
            update_pair<QHALF, ORMODE, SMALLD>(vA, upA, dnA, lfA, rtA, vB, upB, dnB, lfB, rtB, wA0, wA1, wB0, wB1,
                                       hs, hc1, nlT, d.bc, d.bs, renorm, accA, accB);
            S[offA] = vA;
            if (eB != eA) S[offB] = vB;
            if constexpr (FUSED) {
                if (count) n_accepted += (accA && eA < n_core && offA - own_lo < own_span) + (accB && eB != eA && eB < n_core && offB - own_lo < own_span);
            }
        };
        // full rounds: thread tid takes the entries pos + tid and pos + NT + tid; the last round splits what
        // is left into two halves of whole warps, so that no warp runs a round for a missing second site
        auto half_sweep = [&](auto draw_tag) {
            uint32_t pos = 0;
#pragma unroll 1
            for (; pos + 2u * NT <= n; pos += 2u * NT) update_two(draw_tag, pos + tid, pos + NT + tid);
            if (pos < n) {
                const uint32_t stride = ((n - pos + 63u) >> 6) << 5;
                const uint32_t eA = pos + tid;
                if ((uint32_t)tid < stride && eA < n) update_two(draw_tag, eA, eA + stride < n ? eA + stride : eA);
            }
        };
        if (!fresh) half_sweep(DrawTag<DRAW_STORED>{});
        else if (!odd && stash) half_sweep(DrawTag<DRAW_EVEN_STORE>{});
        else half_sweep(DrawTag<DRAW_ANY>{});
        __syncthreads();
        if (h.flags & HS_ACC) {                 // a realization is complete: its state into the sums (reads the core only)
            accumulate_core(st.realizations + real_no + (h.flags >> 16));
            __syncthreads();                    // before the next half-sweep writes core sites
        }
        if constexpr (EQUIL) {
            if ((h.flags >> 8) & 1u) {          // a whole sweep is done (colour 1 was its second half): steps 5.2-5.5
                n_accepted = __reduce_add_sync(0xFFFFFFFFu, n_accepted);
                if (lane == 0 && n_accepted) atomicAdd(&s_accepted, n_accepted);
                n_accepted = 0;
                const double e_warp = core_energy_warp(d, S, tg, H, FC, warp, lane, NW);
                if (lane == 0) s_red[warp] = e_warp;
                __syncthreads();
                if (tid == 0) {
                    double sum = 0.0;
                    for (int w = 0; w < NW; ++w) sum += s_red[w];
                    s_state->accepted = (unsigned long long)s_accepted;
                    s_accepted = 0;
                    controller_step(d, *s_state, -sum);
                    s_ctrl[0] = s_state->hd_scale;
                    s_ctrl[1] = s_state->done ? 1.0f : 0.0f;
                }
                __syncthreads();
                hs = s_ctrl[0]; hc1 = hs * 5.9604644775390625e-08f;
                finished = s_ctrl[1] != 0.0f;
            }
        }
      }
    }
    fence_proxy_async_smem();
    __syncthreads();

    // write the core back, one bulk copy per row (an odd last column takes the zero pad column along)
    const uint32_t row_bytes = (uint32_t)((tg.TCc + 1) & ~1) * (uint32_t)sizeof(float2);
    // rows dealt over the warps first, then over a warp's lanes: the copy engine takes its operands from uniform
    // registers, one issuing lane after the other, so every warp issues its few copies at the same time
    for (int lr = warp + NW * lane; lr < tg.TRc; lr += NW * 32)
        bulk_store(dst + (size_t)(tg.r0 + lr) * d.pitch + tg.c0, S + (H + lr) * FC + H, row_bytes);

    if (FUSED && !EQUIL) {
        if (count) {
            n_accepted = __reduce_add_sync(0xFFFFFFFFu, n_accepted);
            if (lane == 0 && n_accepted) atomicAdd(&s_accepted, n_accepted);
        }
        if (flags & PASS_ENERGY) {
            // a5: H_tile = - sum over the core's colour-1 sites (fixed ones too) of v . h; fixed summation order
            const double sum = core_energy_warp(d, S, tg, H, FC, warp, lane, NW);
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
    if constexpr (EQUIL) {
        // the state goes back: cur = where the row copies above put the vectors, whatever the sweep count
        if (tid == 0) { s_state->cur = src_buf ^ 1u; if (s_state->done) d.done_flags[g] = 1u; }
        __syncthreads();
        for (uint32_t w = tid; w < sizeof(GridState) / 4; w += NT)
            reinterpret_cast<uint32_t*>(&d.states[g])[w] = reinterpret_cast<const uint32_t*>(s_state)[w];
    }
    bulk_commit_wait_read();      // shared memory must stay until the row copies have read it
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
    const float2* v = vec_grid(d, g, d.states[g].cur);
    const float2 zero = make_float2(0.0f, 0.0f);
    double sum = 0.0;
    for (int r = d.own_r0 + blockIdx.x; r < d.own_r1; r += gridDim.x) {
        const float2* row = v + (size_t)r * d.pitch;
        float part = 0.0f;
        int cnt = 0;
        for (int col = ((r + 1) & 1) + 2 * (int)threadIdx.x; col < d.cols; col += 2 * ENERGY_THREADS) {
            const float2 c = row[col];
            const float2 up = r > 0 ? row[col - (int)d.pitch] : zero, dn = r + 1 < d.rows ? row[col + d.pitch] : zero;
            const float2 lf = col > 0 ? row[col - 1] : zero, rt = col + 1 < d.cols ? row[col + 1] : zero;
            part += fmaf(c.x, (up.x + dn.x) + (lf.x + rt.x), c.y * ((up.y + dn.y) + (lf.y + rt.y)));
            if (++cnt == 8) { sum += (double)part; part = 0.0f; cnt = 0; }
        }
        sum += (double)part;
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

// Sum of a grid's n partials by one block of REDUCE_THREADS threads in a fixed order (strided per thread, shuffle
// tree per warp, warps in order): bitwise reproducible.  Every thread of the block must call it; thread 0 gets the sum.
constexpr int REDUCE_THREADS = 256;
__device__ __forceinline__ double sum_energy_partials(const Dev& d, int g, int n)
{
    __shared__ double warp_part[REDUCE_THREADS / 32];
    const double* p = d.e_partials + (size_t)g * d.n_partials;
    double s = 0.0;
    for (int b = threadIdx.x; b < n; b += REDUCE_THREADS) s += p[b];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xFFFFFFFFu, s, o);
    if ((threadIdx.x & 31) == 0) warp_part[threadIdx.x >> 5] = s;
    __syncthreads();
    double total = 0.0;
    if (threadIdx.x == 0)
        for (int w = 0; w < REDUCE_THREADS / 32; ++w) total += warp_part[w];
    return total;
}

__global__ void k_energy_query(Dev d, int n_partials)
{
    const int g = blockIdx.x;
    const double H = sum_energy_partials(d, g, n_partials);
    if (threadIdx.x == 0) d.states[g].e_query = H / d.n_bonds;
}

// ---------------------------------------------------------------------------
// Alg. 2 step 4.1 (Eq. 4): sample specific energy.  Block b sums -cos q(phi_i - phi_j)
// over the bonds (right, down) between SAMPLE sites of its rows in double (fixed order: reproducible);
// the pair count goes through an integer atomic.  k_sample_energy_finish divides.
// ---------------------------------------------------------------------------
__global__ void __launch_bounds__(ENERGY_THREADS) k_sample_energy(Dev d)
{
    const int g = blockIdx.y;
    __shared__ double warp_sum[ENERGY_THREADS / 32];
    const float* phi = d.phi + (size_t)g * d.N;
    const uint32_t* bits = d.bits + (size_t)g * d.words;
    const double q = (double)d.q;
    double sum = 0.0;
    unsigned long long cnt = 0ull;
    for (int r = blockIdx.x; r < d.rows; r += gridDim.x)
        for (int col = threadIdx.x; col < d.cols; col += ENERGY_THREADS) {
            const uint32_t n = (uint32_t)r * d.cols + col;
            if (!is_fixed(bits, n)) continue;
            const double p = (double)phi[n];
            if (col + 1 < d.cols && is_fixed(bits, n + 1)) { sum -= cos(q * (p - (double)phi[n + 1])); ++cnt; }
            if (r + 1 < d.rows && is_fixed(bits, n + d.cols)) { sum -= cos(q * (p - (double)phi[n + d.cols])); ++cnt; }
        }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        sum += __shfl_xor_sync(0xFFFFFFFFu, sum, o);
        cnt += __shfl_xor_sync(0xFFFFFFFFu, cnt, o);
    }
    if ((threadIdx.x & 31) == 0) { warp_sum[threadIdx.x >> 5] = sum; if (cnt) atomicAdd(&d.states[g].n_pairs, cnt); }
    __syncthreads();
    if (threadIdx.x == 0) {
        double s = 0.0;
        for (int w = 0; w < ENERGY_THREADS / 32; ++w) s += warp_sum[w];
        d.e_partials[(size_t)g * d.n_partials + blockIdx.x] = s;
    }
}
__global__ void k_zero_pairs(Dev d)
{
    const int g = blockIdx.x * blockDim.x + threadIdx.x;
    if (g < d.batch) d.states[g].n_pairs = 0ull;
}

// ---------------------------------------------------------------------------
// Alg. 2 step 4.2 (Eq. 5): energy averaged over the sweeps of a chain.  After each
// K = 1 pass with the fused energy reduction: e_sum += H / N_GP, and the sweep is committed.
// ---------------------------------------------------------------------------
__global__ void k_measure_begin(Dev d)
{
    const int g = blockIdx.x * blockDim.x + threadIdx.x;
    if (g < d.batch) { d.states[g].e_sum = 0.0; d.states[g].n_meas = 0u; }
}
__global__ void k_measure(Dev d)
{
    const int g = blockIdx.x;
    GridState& s = d.states[g];
    const double H = sum_energy_partials(d, g, d.ntiles);
    if (threadIdx.x != 0) return;
    s.e_last = H / d.n_bonds;
    s.e_sum += s.e_last; s.n_meas += 1u;
    s.t += 1u; s.cur ^= 1u;
}
__global__ void k_sample_energy_finish(Dev d, int n_partials)
{
    const int g = blockIdx.x;
    const double sum = sum_energy_partials(d, g, n_partials);
    if (threadIdx.x == 0) d.states[g].e_query = d.states[g].n_pairs ? sum / (double)d.states[g].n_pairs : 0.0;
}

// ---------------------------------------------------------------------------
// a6  equilibration controller: Alg. 2 steps 5.2-5.5 for
// one grid per block, after the sweep (5.1) with its fused energy reduction.
// Commits the sweep: t += 1 and the vector buffers swap roles.
// ---------------------------------------------------------------------------
__global__ void k_controller(Dev d)
{
    // launched with programmatic stream serialization behind a fused tile pass: it may be resident before that pass has
    // drained (and lets the next pass load its tile lists meanwhile), but reads nothing before the pass is complete
    griddep_launch_dependents();
    griddep_wait();
    const int g = blockIdx.x;
    GridState& s = d.states[g];
    if (s.done) return;
    const double H = sum_energy_partials(d, g, d.ntiles);
    if (threadIdx.x != 0) return;
    controller_step(d, s, H);
    if (s.done) d.done_flags[g] = 1u;
}

// One grid cut into row blocks over several contexts (mpr_create_slab).  k_slab_partial: this slab's share of the
// sweep's energy (its own rows' colour-1 sites) into e_query; the host adds the slabs' shares and accepted counts and
// k_controller_slab takes steps 5.2-5.5 with the totals -- every slab the same step, since the totals are the same.
__global__ void k_slab_partial(Dev d, int n_partials)
{
    const double H = sum_energy_partials(d, 0, n_partials);
    if (threadIdx.x == 0) d.states[0].e_query = H;
}
__global__ void k_controller_slab(Dev d, double H_total, unsigned long long accepted_total, double P_total)
{
    GridState& s = d.states[0];
    if (s.done) return;
    s.accepted = accepted_total;
    controller_step(d, s, H_total, P_total);
    if (s.done) d.done_flags[0] = 1u;
}
// Eq. 1 range given from outside (the minimum and maximum over every slab's samples)
__global__ void k_set_range(Dev d, float zmin, float zmax)
{
    d.states[0].zmin = zmin; d.states[0].zmax = zmax;
}

// scalar state edits ---------------------------------------------------------
// mode 0: a <- a_value for every grid; mode 1: keep a (refresh the derived scale only)
__global__ void k_set_a(Dev d, int mode, double a_value, int zero_accepted)
{
    const int g = blockIdx.x * blockDim.x + threadIdx.x;
    if (g >= d.nv) return;
    GridState& s = d.states[g];
    if (mode == 0) s.a = a_value;
    s.hd_scale = (float)((double)d.q * (0.5 * (double)TWO_PI_F) / s.a);
    if (zero_accepted) s.accepted = 0ull;
}
// commit passes that ran with (t_off, flip) arguments: t += n_sweeps, swap buffers if the pass count was odd
__global__ void k_commit(Dev d, int first, int n_states, uint32_t n_sweeps, uint32_t flip, uint32_t n_realizations)
{
    const int g = first + blockIdx.x * blockDim.x + threadIdx.x;
    if (g >= first + n_states) return;
    GridState& s = d.states[g];
    s.t += n_sweeps; s.cur ^= flip; s.realizations += n_realizations;
}
// after equilibration: grids whose state sits in buffer 1 are copied into buffer 0 (then k_set_cur(0))
__global__ void __launch_bounds__(256) k_unify_cur(Dev d)
{
    const int g = blockIdx.y;
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < d.VG && d.states[g].cur == 1u) vec_grid(d, g, 0)[i] = vec_grid(d, g, 1)[i];
}
__global__ void k_set_cur(Dev d, uint32_t cur)
{
    const int g = blockIdx.x * blockDim.x + threadIdx.x;
    if (g < d.batch) d.states[g].cur = cur;
}
__global__ void k_set_t(Dev d, uint32_t t)
{
    const int g = blockIdx.x * blockDim.x + threadIdx.x;
    if (g < d.batch) d.states[g].t = t;
}
// Chain parallelism (reading R25): chain c >= 1 of grid g (state v = g + c * batch) starts step 6 from a copy
// of grid g's equilibrated state: vectors (buffer cur) and the scalars of Alg. 2; it keeps its own realization count.
__global__ void __launch_bounds__(256) k_fork_chains(Dev d, uint32_t cur)
{
    const int v = d.batch + blockIdx.y, g = v % d.batch;
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < d.VG) vec_grid(d, v, cur)[i] = vec_grid(d, g, cur)[i];
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        GridState& s = d.states[v];
        const GridState& o = d.states[g];
        s.t = o.t; s.done = o.done; s.cur = cur; s.hd_scale = o.hd_scale; s.neg_log2e_over_T = o.neg_log2e_over_T;
        s.i = o.i; s.a = o.a; s.k = o.k; s.A_last = o.A_last; s.e_last = o.e_last; s.T = o.T;
        s.zmin = o.zmin; s.zmax = o.zmax; s.accepted = 0ull;
    }
}
__global__ void k_begin_run(Dev d, const float* __restrict__ T)
{
    const int g = blockIdx.x * blockDim.x + threadIdx.x;
    if (g >= d.nv) return;
    GridState& s = d.states[g];
    s.t = 0; s.done = 0; s.cur = 0; s.i = 0; s.realizations = 0; s.accepted = 0ull;
    s.a = 1.0; s.k = -1.0; s.A_last = 0.0; s.e_last = 0.0;
    const double Tg = (double)T[g % d.batch];
    s.T = Tg;
    s.neg_log2e_over_T = (float)(-1.4426950408889634 / Tg);
    s.hd_scale = (float)((double)d.q * (0.5 * (double)TWO_PI_F));
    d.done_flags[g] = 0;
}

// ---------------------------------------------------------------------------
// a8  prediction (Alg. 2 step 7, L148, L212) and the statistics of the realizations.  One block per tile: the
// tile's accumulators are in the order of its core entries (k_tilepass, PASS_ACCUMULATE), the entry gives the site.
// WHAT 0: mean angle over the realizations, back-transformed by the inverse of Eq. 1; sample sites return the input
//         value bit for bit.
// WHAT 1: spread (L212): sample standard deviation of the back-transformed values, 0 at sample sites.
// WHAT 2: Gaussian p-quantile from the pooled mean and spread (reading R26): z_p = mean_z + x_p s_z with
//         x_p = Phi^-1(p) computed on the host, clamped to the data range; sample sites = input.
// The realizations of every chain of the grid are pooled (one chain: the paper's step 7): sum of squared deviations
// from the pooled mean = sum over the chains of [their own m2 + n_c (mean_c - mean)^2].
// ---------------------------------------------------------------------------
template <int WHAT>
__global__ void __launch_bounds__(256) k_predict(Dev d, double x_p, float* __restrict__ out)
{
    const int tile = blockIdx.x, g = blockIdx.y;
    const TileGeom tg = tile_geom(d, tile);
    const GridState& s = d.states[g];
    const uint32_t* bits = d.bits + (size_t)g * d.words;
    // sample sites of the core
    for (int i = threadIdx.x; i < tg.TRc * tg.TCc; i += blockDim.x) {
        const int lr = i / tg.TCc, lc = i - lr * tg.TCc;
        const uint32_t n = (uint32_t)(tg.r0 + lr) * d.cols + (uint32_t)(tg.c0 + lc);
        if (is_fixed(bits, n)) out[(size_t)g * d.N + n] = WHAT == 1 ? 0.0f : d.values[(size_t)g * d.N + n];
    }
    // prediction sites: the core entries of both colours
    const TileMeta& meta = d.tile_meta[(size_t)g * d.ntiles + tile];
    const uint16_t* E = d.entries + (size_t)g * d.entry_stride + (size_t)tile * d.tile_entries;
    const uint32_t n0 = meta.cle[0][0], a1 = colour1_base(n0), n_acc = a1 + meta.cle[1][0], e1 = colour1_base(meta.cle[0][MAX_H - 1]);
    const double scale = ((double)s.zmax - (double)s.zmin) / (double)TWO_PI_F;
    for (uint32_t i = threadIdx.x; i < n_acc; i += blockDim.x) {
        if (i >= n0 && i < a1) continue;
        const uint32_t off = E[i < n0 ? i : e1 + (i - a1)];
        const uint32_t lr = off / (uint32_t)d.FC, lc = off - lr * (uint32_t)d.FC;
        const uint32_t n = (uint32_t)(tg.r0 - d.H + (int)lr) * d.cols + (uint32_t)(tg.c0 - d.H + (int)lc);
        MPR_CHECK(n < d.N && i < d.acc_stride && !is_fixed(bits, n));
        double sum = 0.0, count = 0.0;
        for (int c = 0; c < d.chains; ++c) {
            const int v = g + c * d.batch;
            sum += (double)d.acc[((size_t)v * d.ntiles + tile) * d.acc_stride + i]; count += (double)d.states[v].realizations;
        }
        const double mean = sum / count;
        double z;
        if (WHAT == 0) z = (double)s.zmin + mean * scale;
        else {
            double ssd = 0.0;
            for (int c = 0; c < d.chains; ++c) {
                const int v = g + c * d.batch;
                const double nc = (double)d.states[v].realizations;
                if (nc == 0.0) continue;
                const size_t at = ((size_t)v * d.ntiles + tile) * d.acc_stride + i;
                const double dev = (double)d.acc[at] / nc - mean;
                ssd += fmax((double)d.m2[at], 0.0) + nc * dev * dev;
            }
            const double sd = count > 1.0 ? sqrt(ssd / (count - 1.0)) : 0.0;
            if (WHAT == 1) z = sd * scale;
            else z = fmin(fmax((double)s.zmin + mean * scale + x_p * sd * scale, (double)s.zmin), (double)s.zmax);
        }
        out[(size_t)g * d.N + n] = (float)z;
    }
}

// ---------------------------------------------------------------------------
// q learned from the data (reading R28): leave-out validation.
// k_holdout: sample site n is withheld when its uniform of the HOLDOUT stream (Philox counter (n >> 2, 0, 3, g),
// word n & 3) is below `fraction`; train = mask without the withheld samples.
// k_cv_error: sum over the withheld samples of (z - z_hat)^2 in double, fixed block count and summation order.
// ---------------------------------------------------------------------------
struct PhiloxKeys { uint32_t rk0[PHILOX_ROUNDS], rk1[PHILOX_ROUNDS]; };

__global__ void __launch_bounds__(256) k_holdout(PhiloxKeys keys, const uint8_t* __restrict__ mask, uint8_t* __restrict__ train,
                                                 uint8_t* __restrict__ held, uint32_t N, uint32_t g, float fraction)
{
    const uint32_t n = blockIdx.x * blockDim.x + threadIdx.x;
    if (n >= N) return;
    uint8_t h = 0;
    if (mask[n]) {
        const uint4 x = philox4x32_10(n >> 2, 0u, 3u, g, keys.rk0, keys.rk1);
        const uint32_t w = (n & 3u) == 0 ? x.x : (n & 3u) == 1 ? x.y : (n & 3u) == 2 ? x.z : x.w;
        h = u01(w) < fraction ? 1 : 0;
    }
    held[n] = h;
    train[n] = mask[n] && !h ? 1 : 0;
}

__global__ void __launch_bounds__(ENERGY_THREADS) k_cv_error(const float* __restrict__ values, const float* __restrict__ pred,
                                                              const uint8_t* __restrict__ held, uint32_t N,
                                                              double* __restrict__ partials, unsigned long long* __restrict__ count)
{
    __shared__ double warp_sum[ENERGY_THREADS / 32];
    double sum = 0.0;
    unsigned long long cnt = 0ull;
    // block b takes the sites b * chunk .. (b + 1) * chunk - 1 in order: the same sum whatever the device
    const uint32_t chunk = (N + gridDim.x - 1) / gridDim.x, lo = blockIdx.x * chunk, hi = min(N, lo + chunk);
    for (uint32_t n = lo + threadIdx.x; n < hi; n += ENERGY_THREADS)
        if (held[n]) { const double e = (double)values[n] - (double)pred[n]; sum += e * e; ++cnt; }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) { sum += __shfl_xor_sync(0xFFFFFFFFu, sum, o); cnt += __shfl_xor_sync(0xFFFFFFFFu, cnt, o); }
    if ((threadIdx.x & 31) == 0) { warp_sum[threadIdx.x >> 5] = sum; if (cnt) atomicAdd(count, cnt); }
    __syncthreads();
    if (threadIdx.x == 0) {
        double s = 0.0;
        for (int w = 0; w < ENERGY_THREADS / 32; ++w) s += warp_sum[w];
        partials[blockIdx.x] = s;
    }
}
__global__ void k_cv_finish(double* partials, int n)       // one warp: partials[0] <- the sum in a fixed order
{
    double s = 0.0;
    for (int b = threadIdx.x; b < n; b += 32) s += partials[b];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xFFFFFFFFu, s, o);
    if (threadIdx.x == 0) partials[0] = s;
}

// angle import / export at the prediction sites ------------------------------
__global__ void __launch_bounds__(256) k_export_angles(Dev d)
{
    const int g = blockIdx.y;
    const uint32_t n = blockIdx.x * blockDim.x + threadIdx.x;
    if (n >= d.N || is_fixed(d.bits + (size_t)g * d.words, n)) return;
    const uint32_t r = n / d.cols, col = n - r * d.cols;
    const float2 v = vec_grid(d, g, d.states[g].cur)[(size_t)r * d.pitch + col];
    d.phi[(size_t)g * d.N + n] = angle_of(v, d.inv_q);
}
__global__ void __launch_bounds__(256) k_import_angles(Dev d, const float* __restrict__ phi_in)
{
    const int g = blockIdx.y;
    const uint32_t n = blockIdx.x * blockDim.x + threadIdx.x;
    if (n >= d.N || is_fixed(d.bits + (size_t)g * d.words, n)) return;
    const uint32_t r = n / d.cols, col = n - r * d.cols;
    const size_t o = (size_t)g * d.N + n;
    float p = phi_in[o];
    p = p < 0.0f ? 0.0f : p;
    p = p > TWO_PI_F ? TWO_PI_F : p;
    d.phi[o] = p;
    float sn, cs;
    sincosf(__fmul_rn(d.q, p), &sn, &cs);
    vec_grid(d, g, d.states[g].cur)[(size_t)r * d.pitch + col] = make_float2(cs, sn);
}

}  // namespace mpr
