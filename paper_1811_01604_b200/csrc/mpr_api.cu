// mpr_api.cu -- host controller and C ABI (include/mpr.h) of the MPR hot path.
// Everything on the path runs in the kernels of mpr_device.cuh; this file
// validates arguments, lays out the caller's workspace and enqueues launches.
#include "mpr_device.cuh"
#include "mpr_f64.cuh"
#include "../../include/mpr.h"

#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <cudaTypedefs.h>
#include <mutex>
#include <new>
#include <vector>

using namespace mpr;

namespace {

thread_local char g_cuda_err[256] = "";

inline bool cuda_ok(cudaError_t e, const char* what)
{
    if (e == cudaSuccess) return true;
    snprintf(g_cuda_err, sizeof g_cuda_err, "%s: %s", what, cudaGetErrorString(e));
    return false;
}
#define CU(call) do { if (!cuda_ok((call), #call)) return MPR_ERR_CUDA; } while (0)
// this library links its own (static) CUDA runtime, whose current device is not torch's
#define ENTER(ctx) do { if (!cuda_ok(cudaSetDevice((ctx)->device), "cudaSetDevice")) return MPR_ERR_CUDA; } while (0)
#define CU_LAUNCH() do { ++ctx->launches; if (!cuda_ok(cudaGetLastError(), "kernel launch")) return MPR_ERR_CUDA; } while (0)

inline size_t align_up(size_t x, size_t a = 256) { return (x + a - 1) / a * a; }
inline unsigned cdiv(size_t a, size_t b) { return (unsigned)((a + b - 1) / b); }

struct Geometry {
    uint32_t N, words, pitch;
    size_t VG;
    int TR, TC, H, FR, FC, ntx, nty, ntiles;
    uint32_t n_partials, acc_stride;
    size_t entry_stride;
};

// tile passes resident at once on the device this library is written for: 148 SMs x 3 CTAs (B200)
constexpr long RESIDENT_TILE_PASSES = 148L * 3L;

// Tile shape.  A grid that fits one frame is a single tile with a
// two-site zero border (any number of sweeps per pass); otherwise TR x TC cores with a halo of H
// (H/2 sweeps per pass).  TC, H and FC are even so that every core row starts on a 16-byte boundary
// of shared memory (bulk row copies).  (Built with -DMPR_EXPERIMENT_HOOKS, which the shipped library is not,
// MPR_TILE="TR,TC,H" overrides the default.)
void choose_tiles(int batch, int rows, int cols, Geometry* g)
{
    int TR = 64, TC = 64, H = 8;
    // a batch that does not fill the device with 64-row tiles gets lower ones (same frame pitch), as low as still
    // fits one wave: more CTAs in flight, shorter half-sweeps (measured: 256^2 2.7 instead of 4.1 us per sweep)
    const long ntx64 = (cols + 63) / 64;
    if ((long)batch * ntx64 * ((rows + 63) / 64) < RESIDENT_TILE_PASSES) {
        for (int tr = 16; tr < 64; tr += 8)
            if ((long)batch * ntx64 * ((rows + tr - 1) / tr) <= RESIDENT_TILE_PASSES) { TR = tr; break; }
        // still room at 16 rows: narrower tiles too (a pass of such a grid lasts as long as ONE tile's 2K half-sweeps, so
        // halving a tile's sites matters more than the halo it recomputes; measured on 256^2: 64 tiles of 16 x 64 34.2 ms
        // per grid, 128 of 16 x 32 26.3 ms, 256 of 16 x 16 21.9 ms)
        if (TR == 16)
            for (int tc = 32; tc >= 16; tc /= 2) {
                if ((long)batch * ((cols + tc - 1) / tc) * ((rows + 15) / 16) > RESIDENT_TILE_PASSES) break;
                TC = tc;
            }
    }
#ifdef MPR_EXPERIMENT_HOOKS
    if (const char* e = getenv("MPR_TILE")) {
        int a, b, c;
        if (sscanf(e, "%d,%d,%d", &a, &b, &c) == 3 && a >= 8 && b >= 8 && (b & 1) == 0 && c >= 2 && c <= MAX_H &&
            (c & 1) == 0 && (a + 2 * c) * (b + 2 * c + 2) <= 65535 && a + 2 * c <= 255 && b + 2 * c <= 252) { TR = a; TC = b; H = c; }
    }
#endif
    if ((long)rows * cols <= 128L * 128L && rows <= 250 && cols <= 250) { TR = rows; TC = cols; H = 2; }
    g->TR = TR; g->TC = TC; g->H = H; g->FR = TR + 2 * H;
    g->FC = ((TC + 2 * H + 1) & ~3) + 2;        // >= TC + 2H and = 2 (mod 4): a column's rows spread over the banks
    g->ntx = (cols + TC - 1) / TC; g->nty = (rows + TR - 1) / TR; g->ntiles = g->ntx * g->nty;
    g->n_partials = (uint32_t)(g->ntiles > ENERGY_BLOCKS ? g->ntiles : ENERGY_BLOCKS);
    g->acc_stride = (((uint32_t)TR * (uint32_t)TC + 15u) & ~15u) + 16u;   // two 16-aligned runs of core entries per tile
    g->entry_stride = (size_t)g->ntiles * (((size_t)g->FR * g->FC + 31) & ~(size_t)15);   // two 16-aligned lists per tile
}

bool make_geometry(int batch, int chains, int rows, int cols, Geometry* g)
{
    if (batch < 1 || chains < 1 || (long)batch * chains > 65535 || rows < 2 || cols < 2 || rows > 65534 || cols > 65534) return false;
    const uint64_t N = (uint64_t)rows * (uint64_t)cols;
    const uint64_t pitch = ((uint64_t)cols + 1) & ~1ull;                      // even: rows start 16-byte aligned
    if (N >= (1ull << 31) || (uint64_t)rows * pitch >= (1ull << 31)) return false;
    g->N = (uint32_t)N; g->words = (uint32_t)((N + 31) / 32);
    g->pitch = (uint32_t)pitch; g->VG = (size_t)rows * pitch;
    choose_tiles(batch * chains, rows, cols, g);        // step 6 runs every chain of every grid at once
    return g->entry_stride < (1ull << 32);
}

struct Layout {
    size_t states, done, partials, values, phi, bits, vec, acc, m2, tile_meta, entries, total;
};

// B grids with data of their own, V = B * chains states (vectors, accumulators, Alg. 2 scalars)
Layout make_layout(int batch, int chains, const Geometry& g)
{
    Layout L;
    size_t o = 0;
    auto take = [&](size_t bytes) { size_t at = o; o = align_up(o + bytes); return at; };
    const size_t B = (size_t)batch, V = B * (size_t)chains;
    L.states    = take(V * sizeof(GridState));
    L.done      = take(V * sizeof(uint32_t));
    L.partials  = take(B * g.n_partials * sizeof(double));
    L.values    = take(B * g.N * sizeof(float));
    L.phi       = take(B * g.N * sizeof(float));
    L.bits      = take(B * g.words * sizeof(uint32_t));
    L.vec       = take(2 * V * g.VG * sizeof(float2));
    L.acc       = take(V * (size_t)g.ntiles * g.acc_stride * sizeof(float));
    L.m2        = take(V * (size_t)g.ntiles * g.acc_stride * sizeof(float));
    L.tile_meta = take(B * g.ntiles * sizeof(TileMeta));
    L.entries   = take((B * g.entry_stride + 16) * sizeof(uint16_t));
    L.total = o;
    return L;
}

enum RunState { CREATED = 0, READY = 1 };

// ghost rows a slab keeps of each neighbour: the halo of the tile pass, i.e. up to SLAB_GHOST / 2 sweeps between exchanges
constexpr int SLAB_GHOST = 8;

}  // namespace

struct mpr_ctx {
    alignas(64) CUtensorMap map[2][MAX_H / 2 + 1];   // frame boxes of the two vector buffers (TMA descriptors), [buffer][row halo / 2]
    Dev          d;
    Layout       lay;
    cudaStream_t stream;
    mpr_params   prm;
    RunState     state;
    int          energy_blocks;
    uint32_t     k_max;           // sweeps per tile pass
    size_t       smem_bytes;      // dynamic shared memory of k_tilepass
    uint64_t     launches;
    uint32_t*    h_done;          // [batch] host copy of the done flags (pageable: a pinned allocation costs ~1 ms per context)
    GridState*   h_states;        // [batch] pageable host copy
    bool         qhalf;
    bool         dirty;           // vectors changed since d.phi was last written at the free sites
    int          device;          // device the workspace lives on
    bool         no_pdl;          // launch the tile passes without programmatic stream serialization (-DMPR_EXPERIMENT_HOOKS builds only)
    bool         unconditional;   // no data: every node free, ordered start (Alg. 2 step 4.2)
    double       a_min;           // smallest proposal-width parameter a over the grids, as far as the host knows it (0 = unknown)
    bool         small_d;         // every grid's proposal half-rotation q pi / (2 a) is below SMALL_HD (host knowledge of a)
    uint32_t     cur;             // vector buffer holding the current state, the same for every grid outside mpr_equilibrate
    uint32_t     pf_dist[2];      // tile passes resident on the device at once (L2 prefetch distance), 0 = not yet known; [1]: single-sweep passes
    int          active;          // states the tile passes cover: the grids (chain 0), or every chain inside mpr_simulate,
    int          first;           //   or one group of grids (mpr_set_grid_group): states first .. first + active - 1
    int          group;           // grids per group in mpr_simulate (0 = all at once)
    bool         forked;          // chains >= 1 hold a copy of their grid's state (until chain 0 alone moves again)
    uint64_t     n_realizations;  // realizations accumulated per grid (all of its chains) since mpr_set_params
    // one grid cut into row blocks (mpr_create_slab)
    bool         slab;
    mpr_slab     slab_cfg;
    int          ghost_up, ghost_down;   // ghost rows above / below the own rows (SLAB_GHOST, or 0 at the grid's edge)
    double       P_total;                // prediction sites of the whole grid
};

namespace {

mpr_status fetch_states(mpr_ctx* ctx)
{
    CU(cudaMemcpyAsync(ctx->h_states, ctx->d.states, sizeof(GridState) * ctx->d.nv, cudaMemcpyDeviceToHost, ctx->stream));
    CU(cudaStreamSynchronize(ctx->stream));
    return MPR_OK;
}

typedef void (*pass_kernel)(const CUtensorMap, const CUtensorMap, const Dev, uint32_t, uint32_t, uint32_t, uint32_t, uint32_t, uint32_t, uint32_t, uint32_t, uint32_t);

// fused = with the accepted count / energy reduction / done check compiled in (equilibration, counted sweeps);
// std_fc = the frame pitch is the compile-time STD_FC (standard tile shape)
// small_d = every proposal half-rotation is below SMALL_HD (short sin / cos polynomials); only without the fused tails
// MINB = CTAs per SM the kernel is built for (4: single-sweep passes of the standard tile shape)
template <int FCT, bool SMALLD, int MINB>
pass_kernel pick_pass_kernel_fc(bool qhalf, int or_mode)
{
    if (qhalf) return or_mode == 0 ? k_tilepass<true, 0, false, FCT, SMALLD, false, MINB> : or_mode == 1 ? k_tilepass<true, 1, false, FCT, SMALLD, false, MINB> : k_tilepass<true, 2, false, FCT, SMALLD, false, MINB>;
    return or_mode == 0 ? k_tilepass<false, 0, false, FCT, SMALLD, false, MINB> : k_tilepass<false, 2, false, FCT, SMALLD, false, MINB>;
}
template <int FCT, int MINB>
pass_kernel pick_fused_kernel_fc(bool qhalf, int or_mode)
{
    if (qhalf) return or_mode == 0 ? k_tilepass<true, 0, true, FCT, false, false, MINB> : or_mode == 1 ? k_tilepass<true, 1, true, FCT, false, false, MINB> : k_tilepass<true, 2, true, FCT, false, false, MINB>;
    return or_mode == 0 ? k_tilepass<false, 0, true, FCT, false, false, MINB> : k_tilepass<false, 2, true, FCT, false, false, MINB>;
}
// Alg. 2 step 5 inside the pass (grids that are one tile)
template <int FCT>
pass_kernel pick_equil_kernel_fc(bool qhalf, int or_mode)
{
    if (qhalf) return or_mode == 0 ? k_tilepass<true, 0, true, FCT, false, true> : or_mode == 1 ? k_tilepass<true, 1, true, FCT, false, true> : k_tilepass<true, 2, true, FCT, false, true>;
    return or_mode == 0 ? k_tilepass<false, 0, true, FCT, false, true> : k_tilepass<false, 2, true, FCT, false, true>;
}
pass_kernel pick_equil_kernel(bool qhalf, int or_mode, bool std_fc)
{
    return std_fc ? pick_equil_kernel_fc<STD_FC>(qhalf, or_mode) : pick_equil_kernel_fc<0>(qhalf, or_mode);
}
// four = a single-sweep pass of the standard tile shape: the instantiation budgeted for four CTAs per SM
pass_kernel pick_pass_kernel(bool qhalf, int or_mode, bool fused, bool std_fc, bool small_d, bool four = false)
{
    if (four && std_fc) {
        if (fused) return pick_fused_kernel_fc<STD_FC, 4>(qhalf, or_mode);
        return small_d ? pick_pass_kernel_fc<STD_FC, true, 4>(qhalf, or_mode) : pick_pass_kernel_fc<STD_FC, false, 4>(qhalf, or_mode);
    }
    if (fused) return std_fc ? pick_fused_kernel_fc<STD_FC, 3>(qhalf, or_mode) : pick_fused_kernel_fc<0, 3>(qhalf, or_mode);
    if (small_d) return std_fc ? pick_pass_kernel_fc<STD_FC, true, 3>(qhalf, or_mode) : pick_pass_kernel_fc<0, true, 3>(qhalf, or_mode);
    return std_fc ? pick_pass_kernel_fc<STD_FC, false, 3>(qhalf, or_mode) : pick_pass_kernel_fc<0, false, 3>(qhalf, or_mode);
}

void note_a(mpr_ctx* ctx, double a_min)
{
    ctx->a_min = a_min;
    ctx->small_d = a_min > 0.0 && (double)ctx->prm.q * 3.14159265358979323846 / (2.0 * a_min) <= (double)SMALL_HD;
}

// K sweeps (Alg. 1: colour 0, which contains the upper-left node of Fig. 1, then colour 1) of every tile.
// flip = 0 / 1: read buffer ctx->cur ^ flip (known to the host); PER_GRID: each grid reads its own GridState::cur
enum : uint32_t { PER_GRID = 2u };
mpr_status halo_exchange(mpr_ctx* ctx, uint32_t buf);
// acc_every (with PASS_ACCUMULATE): the core is accumulated after every acc_every-th sweep of the pass (0: after the last)
mpr_status launch_pass(mpr_ctx* ctx, uint32_t K, uint32_t t_off, uint32_t flip, uint32_t flags, uint32_t real_no = 0, bool equil = false,
                       uint32_t acc_every = 0)
{
    ctx->dirty = true;
    const bool fused = flags & (PASS_COUNT | PASS_ENERGY | PASS_CHECK_DONE);
    // A pass of K sweeps loads 2K halo rows (a grid that is one tile has its zero border instead of a halo) and, when
    // it is a single sweep, needs no room for stored random words: less shared memory, less to load
    const uint32_t row_halo = ctx->d.ntiles == 1 ? (uint32_t)ctx->d.H : (2u * K < (uint32_t)ctx->d.H ? 2u * K : (uint32_t)ctx->d.H);
    Dev d = ctx->d;
    const bool single = K == 1 && !equil && d.ntiles > 1;
    if (single) d.use_spare = 0;
    const size_t smem = (size_t)(d.TR + 2 * (int)row_halo) * d.FC * sizeof(float2) + (d.use_spare ? 10u : 2u) * (size_t)d.max_entries;
    const pass_kernel kern = equil ? pick_equil_kernel(ctx->qhalf, (int)ctx->prm.or_mode, ctx->d.FC == STD_FC)
                                   : pick_pass_kernel(ctx->qhalf, (int)ctx->prm.or_mode, fused, ctx->d.FC == STD_FC, ctx->small_d, single);
    uint32_t& pf_dist = ctx->pf_dist[single ? 1 : 0];
    if (!pf_dist) {
        int per_sm = 0, sms = 0;
        CU(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, (const void*)kern, TILE_THREADS, smem));
        CU(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, ctx->device));
        pf_dist = (uint32_t)(per_sm > 0 ? per_sm * sms : sms);
#ifdef MPR_EXPERIMENT_HOOKS
        if (const char* e = getenv("MPR_PF_DIST")) pf_dist = (uint32_t)atoi(e) ? (uint32_t)atoi(e) : pf_dist;
#endif
    }
    const uint32_t src_sel = flip == PER_GRID ? PER_GRID : (ctx->cur ^ flip);
    // programmatic stream serialization: this pass's CTAs may start (and load their tile lists) while the last
    // CTAs of the previous kernel still run; k_tilepass waits for that kernel before it reads any result of it
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(ctx->d.ntx, ctx->d.nty, ctx->active); cfg.blockDim = dim3(TILE_THREADS);      // states first .. first + active - 1
    cfg.dynamicSmemBytes = smem; cfg.stream = ctx->stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr; cfg.numAttrs = ctx->no_pdl ? 0 : 1;
    ++ctx->launches;
    const CUtensorMap* maps0 = &ctx->map[0][row_halo / 2], *maps1 = &ctx->map[1][row_halo / 2];
    if (!cuda_ok(cudaLaunchKernelEx(&cfg, kern, *maps0, *maps1, d, K, t_off, src_sel, flags, pf_dist, real_no, row_halo,
                                    (uint32_t)ctx->first, acc_every ? acc_every : K),
                 "tile pass launch")) return MPR_ERR_CUDA;
    return MPR_OK;
}

// n sweeps at the current a as passes of at most k_max sweeps; *t_off and *flip carry the uncommitted progress
mpr_status launch_sweeps(mpr_ctx* ctx, uint32_t n, uint32_t* t_off, uint32_t* flip, uint32_t flags, uint32_t last_flags,
                         uint32_t real_no = 0)
{
    while (n) {
        const uint32_t K = n < ctx->k_max ? n : ctx->k_max;
        mpr_status s = launch_pass(ctx, K, *t_off, *flip, flags | (n == K ? last_flags : 0u), real_no);
        if (s != MPR_OK) return s;
        *t_off += K; *flip ^= 1u; n -= K;
        if (ctx->slab) { s = halo_exchange(ctx, ctx->cur ^ *flip); if (s != MPR_OK) return s; }
    }
    return MPR_OK;
}

// A slab's ghost rows take the neighbouring slabs' rows next to the boundary, as they are in vector buffer `buf`:
// the rows go through the caller's staging buffers, the caller's callback moves them between the slabs.
mpr_status halo_exchange(mpr_ctx* ctx, uint32_t buf)
{
    const Dev& d = ctx->d;
    const mpr_slab& sl = ctx->slab_cfg;
    float2* v = d.vec + (size_t)buf * d.VB;
    const size_t bytes = (size_t)SLAB_GHOST * d.pitch * sizeof(float2);
    if (ctx->ghost_up) CU(cudaMemcpyAsync(sl.d_send_up, v + (size_t)d.own_r0 * d.pitch, bytes, cudaMemcpyDeviceToDevice, ctx->stream));
    if (ctx->ghost_down) CU(cudaMemcpyAsync(sl.d_send_down, v + (size_t)(d.own_r1 - SLAB_GHOST) * d.pitch, bytes, cudaMemcpyDeviceToDevice, ctx->stream));
    if (sl.exchange(sl.user, (void*)ctx->stream)) return MPR_ERR_COMM;
    if (ctx->ghost_up) CU(cudaMemcpyAsync(v, sl.d_recv_up, bytes, cudaMemcpyDeviceToDevice, ctx->stream));
    if (ctx->ghost_down) CU(cudaMemcpyAsync(v + (size_t)d.own_r1 * d.pitch, sl.d_recv_down, bytes, cudaMemcpyDeviceToDevice, ctx->stream));
    return MPR_OK;
}

// Alg. 2 step 5 for one slab of a grid (every slab runs this loop in step): 5.1 one sweep of the own and ghost rows
// with the energy and the accepted proposals of the OWN rows reduced, the ghost rows renewed from the neighbours, 5.3 /
// 5.2 with the sums over the slabs (the caller's all-reduce: two numbers per sweep), 5.4-5.5 on every slab alike.
mpr_status equilibrate_slab(mpr_ctx* ctx)
{
    const Dev& d = ctx->d;
    const mpr_slab& sl = ctx->slab_cfg;
    for (uint32_t i = 0; i < ctx->prm.equil_cap; ++i) {
        mpr_status s = launch_pass(ctx, 1, 0, 0, PASS_COUNT | PASS_ENERGY);
        if (s == MPR_OK) s = halo_exchange(ctx, ctx->cur ^ 1u);
        if (s != MPR_OK) return s;
        k_slab_partial<<<1, REDUCE_THREADS, 0, ctx->stream>>>(d, d.ntiles);
        CU_LAUNCH();
        s = fetch_states(ctx);
        if (s != MPR_OK) return s;
        double sums[2] = {ctx->h_states[0].e_query, (double)ctx->h_states[0].accepted};
        if (sl.allreduce(sl.user, sums, 2, MPR_REDUCE_SUM)) return MPR_ERR_COMM;
        k_controller_slab<<<1, 1, 0, ctx->stream>>>(d, sums[0], (unsigned long long)sums[1], ctx->P_total);
        CU_LAUNCH();
        ctx->cur ^= 1u;                  // the controller committed the sweep: t + 1, the buffers swapped roles
        CU(cudaMemcpyAsync(ctx->h_done, d.done_flags, sizeof(uint32_t), cudaMemcpyDeviceToHost, ctx->stream));
        CU(cudaStreamSynchronize(ctx->stream));
        if (ctx->h_done[0]) break;
    }
    mpr_status s = fetch_states(ctx);
    if (s != MPR_OK) return s;
    note_a(ctx, ctx->h_states[0].a);
    return MPR_OK;
}

// TMA descriptor of one vector buffer: [batch][rows][cols] eight-byte elements with row pitch d.pitch,
// box = one tile frame; elements outside the grid are delivered as zeros (open boundary)
mpr_status make_frame_map(mpr_ctx* ctx, int which, int row_halo)
{
    static PFN_cuTensorMapEncodeTiled encode = nullptr;
    if (!encode) {
        void* fn = nullptr;
        cudaDriverEntryPointQueryResult qres;
        if (!cuda_ok(cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres), "cudaGetDriverEntryPoint") ||
            qres != cudaDriverEntryPointSuccess || !fn) {
            snprintf(g_cuda_err, sizeof g_cuda_err, "cuTensorMapEncodeTiled not available in this driver");
            return MPR_ERR_CUDA;
        }
        encode = (PFN_cuTensorMapEncodeTiled)fn;
    }
    const Dev& d = ctx->d;
    const cuuint64_t dims[3] = {(cuuint64_t)d.cols, (cuuint64_t)d.rows, (cuuint64_t)d.nv};
    const cuuint64_t strides[2] = {(cuuint64_t)d.pitch * sizeof(float2), (cuuint64_t)d.VG * sizeof(float2)};
    const cuuint32_t box[3] = {(cuuint32_t)d.FC, (cuuint32_t)(d.TR + 2 * row_halo), 1u};
    const cuuint32_t estr[3] = {1u, 1u, 1u};
    const CUresult r = encode(&ctx->map[which][row_halo / 2], CU_TENSOR_MAP_DATA_TYPE_UINT64, 3, (void*)(d.vec + (size_t)which * d.VB),
                              dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                              CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) {
        snprintf(g_cuda_err, sizeof g_cuda_err, "cuTensorMapEncodeTiled failed with CUresult %d", (int)r);
        return MPR_ERR_CUDA;
    }
    return MPR_OK;
}

mpr_status launch_energy(mpr_ctx* ctx)
{
    k_energy<<<dim3(ctx->energy_blocks, ctx->d.batch), ENERGY_THREADS, 0, ctx->stream>>>(ctx->d);
    CU_LAUNCH();
    return MPR_OK;
}

dim3 site_grid(const mpr_ctx* ctx) { return dim3(cdiv(ctx->d.N, 256), ctx->d.batch); }

}  // namespace

extern "C" {

const char* mpr_status_string(mpr_status s)
{
    switch (s) {
    case MPR_OK: return "ok";
    case MPR_ERR_ARG: return "bad argument";
    case MPR_ERR_NO_SAMPLES: return "a grid has no sample site";
    case MPR_ERR_NO_FREE: return "a grid has no prediction site";
    case MPR_ERR_DEGENERATE_RANGE: return "sample values have zero range (Eq. 1 divides by zero)";
    case MPR_ERR_NONFINITE: return "a sample value is not finite";
    case MPR_ERR_STATE: return "call out of order";
    case MPR_ERR_WORKSPACE: return "workspace too small or misaligned";
    case MPR_ERR_CUDA: return "CUDA error";
    case MPR_ERR_UNSUPPORTED: return "parameter combination not supported";
    case MPR_ERR_COMM: return "a communication callback of a slab context failed";
    case MPR_ERR_TOO_LARGE: return "size beyond the fixed scratch of the allocation-free entry point";
    }
    return "unknown status";
}

const char* mpr_last_cuda_error(void) { return g_cuda_err; }

void mpr_default_params(mpr_params* p)
{
    if (!p) return;
    memset(p, 0, sizeof *p);
    p->struct_size = (uint32_t)sizeof(mpr_params);
    p->q = 0.5f; p->equil_cap = 500; p->sweeps_per_real = 1; p->M = 100;
    p->n_f = 5; p->n_fit = 20; p->A_targ = 0.3f; p->k_a = 3.0f;
    p->or_mode = 0; p->a_eq_mode = 0; p->seed = 0;
}

mpr_status mpr_query_workspace_chains(int batch, int chains, int rows, int cols, size_t* bytes)
{
    Geometry g;
    if (!bytes || !make_geometry(batch, chains, rows, cols, &g)) return MPR_ERR_ARG;
    *bytes = make_layout(batch, chains, g).total;
    return MPR_OK;
}

mpr_status mpr_query_workspace(int batch, int rows, int cols, size_t* bytes)
{
    return mpr_query_workspace_chains(batch, 1, rows, cols, bytes);
}

}  // extern "C"

namespace {

// mpr_create (data given) and mpr_create_unconditional (d_values = d_sample_mask = nullptr)
// and mpr_create_slab (slab != nullptr: rows = the slab's own rows plus its ghost rows)
mpr_status create_impl(mpr_ctx** out, int batch, int chains, int rows, int cols, const float* d_values,
                       const uint8_t* d_sample_mask, void* d_workspace, size_t workspace_bytes, void* cuda_stream,
                       const mpr_slab* slab = nullptr)
{
    const bool unconditional = !d_values && !d_sample_mask;
    Geometry g;
    if (!out || (!unconditional && (!d_values || !d_sample_mask)) || !make_geometry(batch, chains, rows, cols, &g)) return MPR_ERR_ARG;
    const Layout lay = make_layout(batch, chains, g);
    if (!d_workspace || workspace_bytes < lay.total || ((uintptr_t)d_workspace & 255u)) return MPR_ERR_WORKSPACE;

    mpr_ctx* ctx = new (std::nothrow) mpr_ctx();
    if (!ctx) return MPR_ERR_ARG;
    memset(ctx, 0, sizeof *ctx);
    ctx->lay = lay;
    ctx->stream = (cudaStream_t)cuda_stream;
    {
        cudaPointerAttributes attr;
        if (!cuda_ok(cudaPointerGetAttributes(&attr, d_workspace), "cudaPointerGetAttributes") ||
            attr.type != cudaMemoryTypeDevice) { delete ctx; return MPR_ERR_WORKSPACE; }
        ctx->device = attr.device;
        if (!cuda_ok(cudaSetDevice(ctx->device), "cudaSetDevice")) { delete ctx; return MPR_ERR_CUDA; }
    }
    ctx->state = CREATED;
    ctx->unconditional = unconditional;
#ifdef MPR_EXPERIMENT_HOOKS
    ctx->no_pdl = getenv("MPR_NO_PDL") != nullptr;
#endif
    ctx->prm.q = 0.5f; ctx->d.q = 0.5f; ctx->d.inv_q = 2.0f;      // until mpr_set_params says otherwise (L89)
    char* base = (char*)d_workspace;
    Dev& d = ctx->d;
    d.states = (GridState*)(base + lay.states);
    d.done_flags = (uint32_t*)(base + lay.done);
    d.e_partials = (double*)(base + lay.partials);
    d.values = (float*)(base + lay.values);
    d.phi = (float*)(base + lay.phi);
    d.bits = (uint32_t*)(base + lay.bits);
    d.vec = (float2*)(base + lay.vec);
    d.acc = (float*)(base + lay.acc);
    d.m2 = (float*)(base + lay.m2);
    d.tile_meta = (TileMeta*)(base + lay.tile_meta);
    d.entries = (uint16_t*)(base + lay.entries);
    d.chains = chains; d.nv = batch * chains;
    d.VG = g.VG; d.VB = (size_t)d.nv * g.VG;
    d.entry_stride = g.entry_stride; d.n_partials = g.n_partials; d.acc_stride = g.acc_stride;
    d.tile_entries = (uint32_t)(g.entry_stride / (size_t)g.ntiles);
    d.fc_inv = (uint32_t)(((1u << 24) + (uint32_t)g.FC - 1u) / (uint32_t)g.FC);
    d.TR = g.TR; d.TC = g.TC; d.H = g.H; d.FR = g.FR; d.FC = g.FC; d.ntx = g.ntx; d.nty = g.nty; d.ntiles = g.ntiles;
    d.batch = batch; d.rows = rows; d.cols = cols;
    d.N = g.N; d.words = g.words; d.pitch = g.pitch;
    d.n_bonds = (double)rows * (cols - 1) + (double)cols * (rows - 1);
    d.site_off = 0; d.own_r0 = 0; d.own_r1 = rows;
    if (slab) {
        // rows [row_begin - ghost_up, row_end + ghost_down) of the whole grid; the bonds, the prediction sites and the
        // random streams are those of the whole grid
        ctx->slab = true; ctx->slab_cfg = *slab;
        ctx->ghost_up = slab->row_begin > 0 ? SLAB_GHOST : 0;
        ctx->ghost_down = slab->row_end < slab->rows_global ? SLAB_GHOST : 0;
        d.own_r0 = ctx->ghost_up; d.own_r1 = ctx->ghost_up + (slab->row_end - slab->row_begin);
        d.site_off = (uint32_t)(slab->row_begin - ctx->ghost_up) * (uint32_t)cols;
        d.n_bonds = (double)slab->rows_global * (cols - 1) + (double)cols * (slab->rows_global - 1);
    }
    d.burn_in_only = unconditional ? 1 : 0;
    ctx->energy_blocks = rows < ENERGY_BLOCKS ? rows : ENERGY_BLOCKS;
    ctx->active = batch;
    ctx->h_states = new (std::nothrow) GridState[d.nv];
    mpr_status st = MPR_OK;
    auto fail = [&](mpr_status s) { mpr_destroy(ctx); return s; };
    if (!ctx->h_states) return fail(MPR_ERR_ARG);
    ctx->h_done = new (std::nothrow) uint32_t[batch];
    if (!ctx->h_done) return fail(MPR_ERR_ARG);

    cudaStream_t s = ctx->stream;
    // the pad column of an odd-width grid stays zero
    if (!cuda_ok(cudaMemsetAsync(d.vec, 0, 2 * d.VB * sizeof(float2), s), "memset vec")) return fail(MPR_ERR_CUDA);
    for (int w = 0; w < 2; ++w)
        for (int hr = 2; hr <= g.H; hr += 2) { st = make_frame_map(ctx, w, hr); if (st != MPR_OK) return fail(st); }
    k_state_reset<<<cdiv(d.nv, 128), 128, 0, s>>>(d);
    unsigned mm_blocks = cdiv(g.N, 256 * 8);
    if (mm_blocks > 1184) mm_blocks = 1184;
    if (unconditional) k_state_unconditional<<<cdiv(batch, 128), 128, 0, s>>>(d);
    else if (slab) {
        // Eq. 1's range is over the samples of the WHOLE grid (L81): this slab's own rows, then min / max over the slabs
        k_minmax<<<dim3(mm_blocks, 1), 256, 0, s>>>(d, d_values, d_sample_mask);
        ++ctx->launches;
        st = fetch_states(ctx);
        if (st != MPR_OK) return fail(st);
        const GridState& h = ctx->h_states[0];
        auto decode = [](uint32_t e) { const uint32_t b = (e & 0x80000000u) ? (e & 0x7FFFFFFFu) : ~e; float f; memcpy(&f, &b, sizeof f); return f; };
        const float lo_f = h.n_samples ? decode(h.zmin_enc) : INFINITY;      // the order-preserving encoding of k_minmax
        const float hi_f = h.n_samples ? decode(h.zmax_enc) : -INFINITY;
        double lo = (double)lo_f, hi = (double)hi_f, cnt[2] = {(double)h.n_samples, (h.err_flags & ERRF_NONFINITE) ? 1.0 : 0.0};
        if (slab->allreduce(slab->user, &lo, 1, MPR_REDUCE_MIN) || slab->allreduce(slab->user, &hi, 1, MPR_REDUCE_MAX) ||
            slab->allreduce(slab->user, cnt, 2, MPR_REDUCE_SUM)) return fail(MPR_ERR_COMM);
        if (cnt[0] == 0.0) return fail(MPR_ERR_NO_SAMPLES);
        if (cnt[1] != 0.0) return fail(MPR_ERR_NONFINITE);
        if (!(hi > lo)) return fail(MPR_ERR_DEGENERATE_RANGE);
        k_set_range<<<1, 1, 0, s>>>(d, (float)lo, (float)hi);
    } else {
        k_minmax<<<dim3(mm_blocks, batch), 256, 0, s>>>(d, d_values, d_sample_mask);
        k_minmax_finish<<<cdiv(batch, 128), 128, 0, s>>>(d);
    }
    k_transform<<<dim3(cdiv((size_t)g.words * 32, 256), batch), 256, 0, s>>>(d, d_values, d_sample_mask);
    k_tile_count<<<dim3(g.ntiles, batch), 256, 0, s>>>(d);
    k_tile_scan<<<batch, 32, 0, s>>>(d);
    const size_t fill_smem = (size_t)g.FR * g.FC * sizeof(uint16_t);
    {
        static std::mutex fill_lock;                  // contexts may be created from several host threads
        std::lock_guard<std::mutex> hold(fill_lock);
        static size_t fill_set[64] = {};              // raised only, as for the tile pass below
        size_t& have = fill_set[ctx->device & 63];
        if (fill_smem > 40960 && fill_smem > have) {
            if (!cuda_ok(cudaFuncSetAttribute((const void*)k_tile_fill, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)fill_smem), "k_tile_fill smem"))
                return fail(MPR_ERR_CUDA);
            have = fill_smem;
        }
    }
    // the lists' order: fitted group by group by a serial walk (fewest bank conflicts) when the batch fills the device and
    // the sweeps are bound by throughput; in closed form (k_tile_fill_rounds) when it does not
    if ((long)(batch * chains) * g.ntiles >= RESIDENT_TILE_PASSES) k_tile_fill<<<dim3(g.ntiles, batch), 256, fill_smem, s>>>(d);
    else k_tile_fill_rounds<<<dim3(g.ntiles, batch), 256, 0, s>>>(d);
    ctx->launches += 7;
    if (!cuda_ok(cudaGetLastError(), "create kernels")) return fail(MPR_ERR_CUDA);
    st = fetch_states(ctx);
    if (st != MPR_OK) return fail(st);
    if (slab) {
        // P of Alg. 2 step 5.2 (A = accepted / P) is the whole grid's number of prediction sites
        double P = (double)ctx->h_states[0].n_free[0] + (double)ctx->h_states[0].n_free[1];
        if (slab->allreduce(slab->user, &P, 1, MPR_REDUCE_SUM)) return fail(MPR_ERR_COMM);
        if (P == 0.0) return fail(MPR_ERR_NO_FREE);
        ctx->P_total = P;
    }
    for (int b = 0; b < batch && !slab; ++b) {
        const uint32_t e = ctx->h_states[b].err_flags;
        if (e & ERRF_NO_SAMPLES) return fail(MPR_ERR_NO_SAMPLES);
        if (e & ERRF_NONFINITE) return fail(MPR_ERR_NONFINITE);
        if (e & ERRF_DEGENERATE) return fail(MPR_ERR_DEGENERATE_RANGE);
        if (e & ERRF_NO_FREE) return fail(MPR_ERR_NO_FREE);
    }
    // shared memory of the tile pass: frame + entries (+ the odd sweeps' random words when they fit)
    uint32_t max_entries = 0;
    for (int b = 0; b < batch; ++b)
        if (ctx->h_states[b].max_tile_entries > max_entries) max_entries = ctx->h_states[b].max_tile_entries;
    max_entries = (max_entries + 15u) & ~15u;
    d.max_entries = max_entries;
    const size_t frame_bytes = (size_t)g.FR * g.FC * sizeof(float2);
    int smem_max = 0;
    if (!cuda_ok(cudaDeviceGetAttribute(&smem_max, cudaDevAttrMaxSharedMemoryPerBlockOptin, ctx->device), "smem attr")) return fail(MPR_ERR_CUDA);
    const size_t budget = (size_t)smem_max - 4096;               // static shared memory of the kernel (2.7 KB with the state copy of k_tilepass<EQUIL>)
    d.use_spare = g.ntiles == 1 || g.H >= 4;                       // pointless when every pass is a single sweep
    if (frame_bytes + 10ull * max_entries > budget) d.use_spare = 0;
    ctx->smem_bytes = frame_bytes + (d.use_spare ? 10ull : 2ull) * max_entries;
    if (ctx->smem_bytes > budget) return fail(MPR_ERR_WORKSPACE);
    ctx->k_max = g.ntiles == 1 ? 1024u : (uint32_t)(g.H / 2);        // mpr_set_pass_depth lowers it (diagnostic)
    if (slab && ctx->k_max > (uint32_t)(SLAB_GHOST / 2)) ctx->k_max = SLAB_GHOST / 2;      // the ghost rows last SLAB_GHOST / 2 sweeps
    // The attribute belongs to the kernel, not to this context: it is only ever raised (per device and frame-pitch
    // variant), so that a context created later with smaller tiles does not take the room of an earlier one away.
    {
        static std::mutex attr_lock;                  // contexts may be created from several host threads
        std::lock_guard<std::mutex> hold(attr_lock);
        static size_t attr_set[64][2] = {};
        size_t& have = attr_set[ctx->device & 63][g.FC == STD_FC ? 1 : 0];
        if (ctx->smem_bytes > have) {
            for (int qh = 0; qh < 2; ++qh)
                for (int om = 0; om < 3; ++om)
                    for (int fu = 0; fu < 2; ++fu)
                        for (int sd = 0; sd < 2; ++sd) {
                            if (!qh && om == 1) continue;
                            if (!cuda_ok(cudaFuncSetAttribute((const void*)pick_pass_kernel(qh, om, fu, g.FC == STD_FC, sd), cudaFuncAttributeMaxDynamicSharedMemorySize,
                                                              (int)ctx->smem_bytes), "cudaFuncSetAttribute")) return fail(MPR_ERR_CUDA);
                            if (g.FC == STD_FC &&
                                !cuda_ok(cudaFuncSetAttribute((const void*)pick_pass_kernel(qh, om, fu, true, sd, true), cudaFuncAttributeMaxDynamicSharedMemorySize,
                                                              (int)ctx->smem_bytes), "cudaFuncSetAttribute")) return fail(MPR_ERR_CUDA);
                            if (fu && !sd &&
                                !cuda_ok(cudaFuncSetAttribute((const void*)pick_equil_kernel(qh, om, g.FC == STD_FC), cudaFuncAttributeMaxDynamicSharedMemorySize,
                                                              (int)ctx->smem_bytes), "cudaFuncSetAttribute")) return fail(MPR_ERR_CUDA);
                        }
            have = ctx->smem_bytes;
        }
    }
    *out = ctx;
    return MPR_OK;
}

}  // namespace

extern "C" {

mpr_status mpr_create(mpr_ctx** out, int batch, int rows, int cols, const float* d_values,
                      const uint8_t* d_sample_mask, void* d_workspace, size_t workspace_bytes, void* cuda_stream)
{
    if (!d_values || !d_sample_mask) return MPR_ERR_ARG;
    return create_impl(out, batch, 1, rows, cols, d_values, d_sample_mask, d_workspace, workspace_bytes, cuda_stream);
}

mpr_status mpr_create_chains(mpr_ctx** out, int batch, int chains, int rows, int cols, const float* d_values,
                             const uint8_t* d_sample_mask, void* d_workspace, size_t workspace_bytes, void* cuda_stream)
{
    if (!d_values || !d_sample_mask) return MPR_ERR_ARG;
    return create_impl(out, batch, chains, rows, cols, d_values, d_sample_mask, d_workspace, workspace_bytes, cuda_stream);
}

mpr_status mpr_create_unconditional(mpr_ctx** out, int batch, int rows, int cols,
                                    void* d_workspace, size_t workspace_bytes, void* cuda_stream)
{
    return create_impl(out, batch, 1, rows, cols, nullptr, nullptr, d_workspace, workspace_bytes, cuda_stream);
}

size_t mpr_slab_halo_bytes(int cols)
{
    return cols < 2 ? 0 : (size_t)SLAB_GHOST * (size_t)((cols + 1) & ~1) * sizeof(float2);
}

static bool slab_ok(const mpr_slab* sl)
{
    return sl && sl->struct_size == sizeof(mpr_slab) && sl->allreduce && sl->exchange && sl->cols >= 2 && sl->rows_global >= 2 &&
           sl->row_begin >= 0 && sl->row_end <= sl->rows_global && (sl->row_begin & 1) == 0 &&
           sl->row_end - sl->row_begin >= SLAB_GHOST && (uint64_t)sl->rows_global * (uint64_t)sl->cols < (1ull << 32) &&
           (sl->row_begin == 0 || (sl->d_send_up && sl->d_recv_up)) && (sl->row_end == sl->rows_global || (sl->d_send_down && sl->d_recv_down));
}

mpr_status mpr_slab_local_rows(const mpr_slab* sl, int* h_first_row, int* h_n_rows)
{
    if (!sl || !h_first_row || !h_n_rows || sl->struct_size != sizeof(mpr_slab) || sl->row_begin < 0 || sl->row_end > sl->rows_global ||
        sl->row_end <= sl->row_begin) return MPR_ERR_ARG;
    const int up = sl->row_begin > 0 ? SLAB_GHOST : 0, down = sl->row_end < sl->rows_global ? SLAB_GHOST : 0;
    if (sl->row_begin - up < 0 || sl->row_end + down > sl->rows_global) return MPR_ERR_ARG;
    *h_first_row = sl->row_begin - up; *h_n_rows = sl->row_end - sl->row_begin + up + down;
    return MPR_OK;
}

mpr_status mpr_query_workspace_slab(const mpr_slab* sl, size_t* bytes)
{
    int first, n;
    if (!bytes || mpr_slab_local_rows(sl, &first, &n) != MPR_OK) return MPR_ERR_ARG;
    return mpr_query_workspace(1, n, sl->cols, bytes);
}

mpr_status mpr_create_slab(mpr_ctx** out, const mpr_slab* sl, const float* d_values, const uint8_t* d_sample_mask,
                           void* d_workspace, size_t workspace_bytes, void* cuda_stream)
{
    int first, n;
    if (!d_values || !d_sample_mask || mpr_slab_local_rows(sl, &first, &n) != MPR_OK || !slab_ok(sl)) return MPR_ERR_ARG;
    return create_impl(out, 1, 1, n, sl->cols, d_values, d_sample_mask, d_workspace, workspace_bytes, cuda_stream, sl);
}

mpr_status mpr_destroy(mpr_ctx* ctx)
{
    if (!ctx) return MPR_ERR_ARG;
    delete[] ctx->h_done;
    delete[] ctx->h_states;
    delete ctx;
    return MPR_OK;
}

mpr_status mpr_set_params(mpr_ctx* ctx, const mpr_params* p, const float* h_T)
{
    if (!ctx || !p || !h_T || p->struct_size != sizeof(mpr_params)) return MPR_ERR_ARG;
    ENTER(ctx);
    if (!(p->q > 0.0f && p->q <= 0.5f) || p->M < 1 || p->sweeps_per_real < 1 || p->n_f < 1 ||
        p->n_fit < 2 || p->n_fit > (uint32_t)MAX_NFIT || !(p->k_a > 0.0f) || !std::isfinite(p->A_targ) ||
        p->or_mode > 2 || p->a_eq_mode > 1)
        return MPR_ERR_ARG;
    for (int b = 0; b < ctx->d.batch; ++b)
        if (!(h_T[b] > 0.0f) || !std::isfinite(h_T[b])) return MPR_ERR_ARG;
    if (p->or_mode == 1 && p->q != 0.5f) return MPR_ERR_UNSUPPORTED;
    ctx->prm = *p;
    ctx->qhalf = p->q == 0.5f;
    Dev& d = ctx->d;
    for (int r = 0; r < PHILOX_ROUNDS; ++r) {          // Philox4x32 key schedule (Weyl sequence)
        d.rk0[r] = (uint32_t)p->seed + (uint32_t)r * 0x9E3779B9u;
        d.rk1[r] = (uint32_t)(p->seed >> 32) + (uint32_t)r * 0xBB67AE85u;
    }
    d.q = p->q; d.inv_q = 1.0f / p->q;
    d.bc = (float)cos((double)p->q * (double)TWO_PI_F); d.bs = (float)sin((double)p->q * (double)TWO_PI_F);
    d.n_f = p->n_f; d.n_fit = p->n_fit; d.equil_cap = p->equil_cap;
    d.A_targ = (double)p->A_targ; d.k_a = (double)p->k_a;
    // per-grid temperatures: staged through the energy partials (free between calls)
    CU(cudaMemcpyAsync(d.e_partials, h_T, sizeof(float) * d.batch, cudaMemcpyHostToDevice, ctx->stream));
    k_begin_run<<<cdiv(d.nv, 128), 128, 0, ctx->stream>>>(d, (const float*)d.e_partials);
    CU_LAUNCH();
    CU(cudaMemsetAsync(d.acc, 0, (size_t)d.nv * d.ntiles * d.acc_stride * sizeof(float), ctx->stream));
    CU(cudaMemsetAsync(d.m2, 0, (size_t)d.nv * d.ntiles * d.acc_stride * sizeof(float), ctx->stream));
    k_init_state<<<dim3(cdiv(d.N, 256), d.batch), 256, 0, ctx->stream>>>(d, ctx->unconditional ? 1 : 0);
    CU_LAUNCH();
    CU(cudaStreamSynchronize(ctx->stream));      // h_T may be pageable and reused by the caller
    ctx->state = READY;
    ctx->dirty = false;
    ctx->cur = 0;
    ctx->forked = false;
    ctx->n_realizations = 0;
    note_a(ctx, 1.0);
    return MPR_OK;
}

mpr_status mpr_equilibrate(mpr_ctx* ctx)
{
    if (!ctx) return MPR_ERR_ARG;
    ENTER(ctx);
    if (ctx->state != READY) return MPR_ERR_STATE;
    const Dev& d = ctx->d;
    ctx->forked = false;           // chain 0 of every grid moves alone (Alg. 2 step 5 is one chain per grid)
    if (ctx->slab) return equilibrate_slab(ctx);
    const uint32_t cap = ctx->prm.equil_cap;
    uint32_t issued = 0;
    auto all_done = [&](bool* all) -> mpr_status {
        CU(cudaMemcpyAsync(ctx->h_done, d.done_flags, sizeof(uint32_t) * d.batch, cudaMemcpyDeviceToHost, ctx->stream));
        CU(cudaStreamSynchronize(ctx->stream));
        *all = true;
        for (int b = 0; b < d.batch; ++b) *all = *all && ctx->h_done[b];
        return MPR_OK;
    };
    if (d.ntiles == 1) {
        // grids that are one tile: steps 5.1-5.5 of up to k_max sweeps in ONE launch per grid batch (k_tilepass<EQUIL>)
        while (issued < cap) {
            const uint32_t K = cap - issued < ctx->k_max ? cap - issued : ctx->k_max;
            mpr_status s = launch_pass(ctx, K, 0, PER_GRID, PASS_COUNT | PASS_ENERGY | PASS_CHECK_DONE, 0, true);
            if (s != MPR_OK) return s;
            issued += K;
            bool all = false;
            s = all_done(&all);
            if (s != MPR_OK) return s;
            if (all) break;
        }
    } else {
        // The controller checks the slope after the sweep with index i when i >= n_fit and i % n_f == 0 (step 5.4), so
        // a grid can only stop after i + 1 sweeps with i such an index: the host polls the flags exactly there.
        const uint32_t n_f = ctx->prm.n_f;
        uint32_t chunk = (ctx->prm.n_fit + n_f - 1) / n_f * n_f + 1;
        while (issued < cap) {
            if (chunk > cap - issued) chunk = cap - issued;
            for (uint32_t j = 0; j < chunk; ++j) {
                // 5.1 one sweep with the energy (5.3) and the accepted count fused; the controller does
                // 5.2, 5.4, 5.5 and commits the sweep (t, buffer swap) for the grids still running
                mpr_status s = launch_pass(ctx, 1, 0, PER_GRID, PASS_COUNT | PASS_ENERGY | PASS_CHECK_DONE);
                if (s != MPR_OK) return s;
                cudaLaunchConfig_t cfg = {};
                cfg.gridDim = dim3(d.batch); cfg.blockDim = dim3(REDUCE_THREADS); cfg.stream = ctx->stream;
                cudaLaunchAttribute attr[1];
                attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
                attr[0].val.programmaticStreamSerializationAllowed = 1;
                cfg.attrs = attr; cfg.numAttrs = ctx->no_pdl ? 0 : 1;
                ++ctx->launches;
                if (!cuda_ok(cudaLaunchKernelEx(&cfg, k_controller, d), "controller launch")) return MPR_ERR_CUDA;
            }
            issued += chunk;
            bool all = false;
            mpr_status s = all_done(&all);
            if (s != MPR_OK) return s;
            if (all) break;
            chunk = n_f;
        }
    }
    // the grids stopped after different numbers of sweeps: bring every state into the same vector buffer
    mpr_status fs = fetch_states(ctx);
    if (fs != MPR_OK) return fs;
    bool any0 = false, any1 = false;
    double a_min = ctx->h_states[0].a;
    for (int b = 0; b < d.batch; ++b) {
        (ctx->h_states[b].cur ? any1 : any0) = true;
        if (ctx->h_states[b].a < a_min) a_min = ctx->h_states[b].a;
    }
    note_a(ctx, a_min);
    if (any0 && any1) {
        k_unify_cur<<<dim3(cdiv(d.VG, 256), d.batch), 256, 0, ctx->stream>>>(d);
        CU_LAUNCH();
        k_set_cur<<<cdiv(d.batch, 128), 128, 0, ctx->stream>>>(d, 0u);
        CU_LAUNCH();
        ctx->cur = 0;
    } else ctx->cur = any1 ? 1u : 0u;
    return MPR_OK;
}

mpr_status mpr_simulate(mpr_ctx* ctx)
{
    if (!ctx) return MPR_ERR_ARG;
    ENTER(ctx);
    if (ctx->state != READY) return MPR_ERR_STATE;
    const Dev& d = ctx->d;
    const uint32_t s_per = ctx->prm.sweeps_per_real;
    k_set_a<<<cdiv(d.nv, 128), 128, 0, ctx->stream>>>(d, ctx->prm.a_eq_mode == 1 ? 0 : 1, 1.0, 0);
    CU_LAUNCH();
    if (ctx->prm.a_eq_mode == 1) note_a(ctx, 1.0);
    // several chains per grid (reading R25): the others start from a copy of chain 0's state, every chain makes
    // ceil(M / chains) realizations, all chains of all grids in the same launches
    uint32_t n_real = ctx->prm.M;
    if (d.chains > 1) {
        if (!ctx->forked) {
            k_fork_chains<<<dim3(cdiv(d.VG, 256), d.nv - d.batch), 256, 0, ctx->stream>>>(d, ctx->cur);
            CU_LAUNCH();
            ctx->forked = true;
        }
        n_real = (ctx->prm.M + (uint32_t)d.chains - 1u) / (uint32_t)d.chains;
        ctx->active = d.nv;
    }
    // One group of grids after the other (mpr_set_grid_group; one chain per grid only): a group's vectors stay in L2
    // from pass to pass when they fit.  Every group does the same passes, so t_off and flip end alike.
    const int group = (ctx->group > 0 && d.chains == 1 && ctx->group < d.batch) ? ctx->group : ctx->active;
    const int n_states = ctx->active;
    uint32_t t_off = 0, flip = 0;
    mpr_status s = MPR_OK;
    for (int g0 = 0; g0 < n_states && s == MPR_OK; g0 += group) {
        ctx->first = g0; ctx->active = n_states - g0 < group ? n_states - g0 : group;
        t_off = 0; flip = 0;
        if (s_per < ctx->k_max) {
            // realizations of fewer sweeps than a pass holds (the paper's s = 1, L210): several of them per launch, the
            // core accumulated inside the pass after every s_per-th sweep (step 6.3)
            const uint32_t per_pass = ctx->k_max / s_per;
            for (uint32_t j = 0; j < n_real && s == MPR_OK; j += per_pass) {
                const uint32_t r = n_real - j < per_pass ? n_real - j : per_pass, K = r * s_per;
                s = launch_pass(ctx, K, t_off, flip, PASS_ACCUMULATE, j + 1u, false, s_per);
                t_off += K; flip ^= 1u;
                if (s == MPR_OK && ctx->slab) s = halo_exchange(ctx, ctx->cur ^ flip);
            }
        } else {
            for (uint32_t j = 0; j < n_real && s == MPR_OK; ++j)
                // s sweeps, the last pass also accumulates phi at the prediction sites (step 6.3)
                s = launch_sweeps(ctx, s_per, &t_off, &flip, 0, PASS_ACCUMULATE, j + 1u);   // realization number: realizations so far + j + 1
        }
    }
    ctx->first = 0; ctx->active = d.batch;
    if (s != MPR_OK) return s;
    k_commit<<<cdiv(d.nv, 128), 128, 0, ctx->stream>>>(d, 0, d.chains > 1 ? d.nv : d.batch, t_off, flip, n_real);
    CU_LAUNCH();
    ctx->cur ^= flip;
    ctx->n_realizations += (uint64_t)n_real * (uint64_t)d.chains;
    return MPR_OK;
}

mpr_status mpr_predict(mpr_ctx* ctx, float* d_out)
{
    if (!ctx || !d_out) return MPR_ERR_ARG;
    ENTER(ctx);
    if (ctx->state != READY || ctx->n_realizations == 0) return MPR_ERR_STATE;     // the mean of no realization is 0 / 0
    const Dev& d = ctx->d;
    k_predict<0><<<dim3(d.ntiles, d.batch), 256, 0, ctx->stream>>>(d, 0.0, d_out);
    CU_LAUNCH();
    return MPR_OK;
}

mpr_status mpr_predict_std(mpr_ctx* ctx, float* d_out)
{
    if (!ctx || !d_out) return MPR_ERR_ARG;
    ENTER(ctx);
    if (ctx->state != READY) return MPR_ERR_STATE;
    mpr_status s = fetch_states(ctx);
    if (s != MPR_OK) return s;
    for (int b = 0; b < ctx->d.batch; ++b) {
        uint32_t n = 0;
        for (int c = 0; c < ctx->d.chains; ++c) n += ctx->h_states[b + c * ctx->d.batch].realizations;
        if (n < 2u) return MPR_ERR_STATE;
    }
    k_predict<1><<<dim3(ctx->d.ntiles, ctx->d.batch), 256, 0, ctx->stream>>>(ctx->d, 0.0, d_out);
    CU_LAUNCH();
    return MPR_OK;
}

mpr_status mpr_predict_quantile(mpr_ctx* ctx, double p, float* d_out)
{
    if (!ctx || !d_out || !(p > 0.0 && p < 1.0)) return MPR_ERR_ARG;
    ENTER(ctx);
    if (ctx->state != READY) return MPR_ERR_STATE;
    mpr_status s = fetch_states(ctx);
    if (s != MPR_OK) return s;
    for (int b = 0; b < ctx->d.batch; ++b) {
        uint32_t n = 0;
        for (int c = 0; c < ctx->d.chains; ++c) n += ctx->h_states[b + c * ctx->d.batch].realizations;
        if (n < 2u) return MPR_ERR_STATE;
    }
    // x_p = Phi^-1(p): the root of erfc(-x / sqrt 2) / 2 = p by bisection (host, once per call)
    double lo = -40.0, hi = 40.0;
    for (int it = 0; it < 200; ++it) {
        const double mid = 0.5 * (lo + hi);
        (0.5 * std::erfc(-mid / std::sqrt(2.0)) < p ? lo : hi) = mid;
    }
    k_predict<2><<<dim3(ctx->d.ntiles, ctx->d.batch), 256, 0, ctx->stream>>>(ctx->d, 0.5 * (lo + hi), d_out);
    CU_LAUNCH();
    return MPR_OK;
}

mpr_status mpr_sample_energy(mpr_ctx* ctx, double* h_e_s, uint64_t* h_n_pairs)
{
    if (!ctx || !h_e_s || !h_n_pairs) return MPR_ERR_ARG;
    ENTER(ctx);
    const Dev& d = ctx->d;
    k_zero_pairs<<<cdiv(d.batch, 128), 128, 0, ctx->stream>>>(d);
    CU_LAUNCH();
    k_sample_energy<<<dim3(ctx->energy_blocks, d.batch), ENERGY_THREADS, 0, ctx->stream>>>(d);
    CU_LAUNCH();
    k_sample_energy_finish<<<d.batch, REDUCE_THREADS, 0, ctx->stream>>>(d, ctx->energy_blocks);
    CU_LAUNCH();
    mpr_status s = fetch_states(ctx);
    if (s != MPR_OK) return s;
    for (int b = 0; b < d.batch; ++b) { h_e_s[b] = ctx->h_states[b].e_query; h_n_pairs[b] = ctx->h_states[b].n_pairs; }
    return MPR_OK;
}

mpr_status mpr_measure_energy(mpr_ctx* ctx, uint32_t n_sweeps, double* h_e_mean)
{
    if (!ctx || !h_e_mean || n_sweeps == 0) return MPR_ERR_ARG;
    ENTER(ctx);
    if (ctx->state != READY) return MPR_ERR_STATE;
    const Dev& d = ctx->d;
    ctx->forked = false;
    k_measure_begin<<<cdiv(d.batch, 128), 128, 0, ctx->stream>>>(d);
    CU_LAUNCH();
    for (uint32_t j = 0; j < n_sweeps; ++j) {
        // one sweep with the energy reduction fused; k_measure adds e and commits the sweep (t, buffer swap)
        mpr_status s = launch_pass(ctx, 1, 0, PER_GRID, PASS_ENERGY);
        if (s != MPR_OK) return s;
        k_measure<<<d.batch, REDUCE_THREADS, 0, ctx->stream>>>(d);
        CU_LAUNCH();
    }
    ctx->cur ^= n_sweeps & 1u;          // every grid swapped buffers n_sweeps times
    mpr_status s = fetch_states(ctx);
    if (s != MPR_OK) return s;
    for (int b = 0; b < d.batch; ++b) h_e_mean[b] = ctx->h_states[b].e_sum / (double)ctx->h_states[b].n_meas;
    return MPR_OK;
}

mpr_status mpr_energy_table(int rows, int cols, const mpr_params* h_params, const float* h_T, int n_T,
                            uint32_t n_meas, void* d_workspace, size_t workspace_bytes, void* cuda_stream,
                            double* h_e)
{
    if (!h_params || !h_T || !h_e || n_T < 1 || n_meas == 0) return MPR_ERR_ARG;
    mpr_ctx* ctx = nullptr;
    mpr_status s = mpr_create_unconditional(&ctx, n_T, rows, cols, d_workspace, workspace_bytes, cuda_stream);
    if (s != MPR_OK) return s;
    s = mpr_set_params(ctx, h_params, h_T);
    if (s == MPR_OK) s = mpr_equilibrate(ctx);
    if (s == MPR_OK) s = mpr_measure_energy(ctx, n_meas, h_e);
    mpr_destroy(ctx);
    return s;
}

mpr_status mpr_infer_temperature(const float* h_T, const double* h_e, int n_T, double e_s, double* h_T_hat)
{
    if (!h_T || !h_e || !h_T_hat || n_T < 1 || !std::isfinite(e_s)) return MPR_ERR_ARG;
    for (int k = 0; k + 1 < n_T; ++k) {
        if (!(h_T[k + 1] > h_T[k])) return MPR_ERR_ARG;
        const double lo = h_e[k], hi = h_e[k + 1];
        if (hi != lo && e_s >= (lo < hi ? lo : hi) && e_s <= (lo < hi ? hi : lo)) {
            *h_T_hat = (double)h_T[k] + (e_s - lo) / (hi - lo) * ((double)h_T[k + 1] - (double)h_T[k]);
            return MPR_OK;
        }
    }
    int best = 0;
    for (int k = 1; k < n_T; ++k)
        if (std::fabs(h_e[k] - e_s) < std::fabs(h_e[best] - e_s)) best = k;
    *h_T_hat = (double)h_T[best];
    return MPR_OK;
}

mpr_status mpr_default_ladder(int rows, int cols, double e_s, const float* h_factors, int n_T, float* h_T)
{
    if (rows < 2 || cols < 2 || !h_T || n_T < 1 || !std::isfinite(e_s)) return MPR_ERR_ARG;
    static const float standard[5] = {0.25f, 0.5f, 1.0f, 2.0f, 4.0f};
    if (!h_factors) { if (n_T != 5) return MPR_ERR_ARG; h_factors = standard; }
    for (int k = 0; k < n_T; ++k)
        if (!(h_factors[k] > 0.0f) || !std::isfinite(h_factors[k]) || (k && !(h_factors[k] > h_factors[k - 1]))) return MPR_ERR_ARG;
    // low-temperature equipartition, e(T) = -1 + (N - 1) T / (2 N_GP): N - 1 harmonic modes of T / 2 each over
    // N_GP bonds (J = 1; reading R15).  Its crossing with e_s only centres the ladder.
    const double n_gp = (double)rows * (cols - 1) + (double)cols * (rows - 1);
    double centre = 2.0 * n_gp * (1.0 + e_s) / ((double)rows * (double)cols - 1.0);
    if (!(centre > 1e-12)) centre = 1e-12;
    for (int k = 0; k < n_T; ++k) h_T[k] = (float)(centre * (double)h_factors[k]);
    return MPR_OK;
}

mpr_status mpr_infer_temperature_auto(mpr_ctx* ctx, const mpr_params* h_params, const float* h_factors, int n_T,
                                      uint32_t n_meas, void* d_workspace, size_t workspace_bytes,
                                      double* h_T_hat, double* h_e_s)
{
    if (!ctx || !h_params || !h_T_hat || n_T < 1 || n_T > 4096 || n_meas == 0) return MPR_ERR_ARG;
    const int batch = ctx->d.batch, rows = ctx->d.rows, cols = ctx->d.cols;
    std::vector<double> e_s, table, T_hat;
    std::vector<uint64_t> pairs;
    std::vector<float> ladder;
    try {
        e_s.resize((size_t)batch); table.resize((size_t)n_T); T_hat.resize((size_t)batch);
        pairs.resize((size_t)batch); ladder.resize((size_t)n_T);
    } catch (...) { return MPR_ERR_ARG; }
    // step 4.1 with the q of h_params: Eq. 4 depends on q only through cos q(phi_i - phi_j)
    const float q_keep = ctx->d.q;
    if (!(h_params->q > 0.0f && h_params->q <= 0.5f)) return MPR_ERR_ARG;
    ctx->d.q = h_params->q;
    mpr_status s = mpr_sample_energy(ctx, e_s.data(), pairs.data());
    ctx->d.q = q_keep;
    if (s != MPR_OK) return s;
    for (int g = 0; g < batch; ++g) {
        if (pairs[(size_t)g] == 0) return MPR_ERR_NO_SAMPLES;       // no pair of neighbouring samples: e_s is undefined
        s = mpr_default_ladder(rows, cols, e_s[(size_t)g], h_factors, n_T, ladder.data());
        if (s == MPR_OK) s = mpr_energy_table(rows, cols, h_params, ladder.data(), n_T, n_meas, d_workspace, workspace_bytes,
                                              (void*)ctx->stream, table.data());
        if (s == MPR_OK) s = mpr_infer_temperature(ladder.data(), table.data(), n_T, e_s[(size_t)g], &T_hat[(size_t)g]);
        if (s != MPR_OK) return s;
    }
    for (int g = 0; g < batch; ++g) { h_T_hat[g] = T_hat[(size_t)g]; if (h_e_s) h_e_s[g] = e_s[(size_t)g]; }
    return MPR_OK;
}

namespace {
struct LearnLayout { size_t ctx, train, held, pred, partials, count, total; };
bool learn_layout(int rows, int cols, LearnLayout* L)
{
    size_t ws = 0;
    if (mpr_query_workspace(1, rows, cols, &ws) != MPR_OK) return false;
    const size_t N = (size_t)rows * cols;
    size_t o = 0;
    auto take = [&](size_t bytes) { size_t at = o; o = align_up(o + bytes); return at; };
    L->ctx = take(ws); L->train = take(N); L->held = take(N); L->pred = take(N * sizeof(float));
    L->partials = take(ENERGY_BLOCKS * sizeof(double)); L->count = take(sizeof(unsigned long long));
    L->total = o;
    return true;
}
}  // namespace

mpr_status mpr_query_workspace_learn_q(int rows, int cols, size_t* bytes)
{
    LearnLayout L;
    if (!bytes || !learn_layout(rows, cols, &L)) return MPR_ERR_ARG;
    *bytes = L.total;
    return MPR_OK;
}

mpr_status mpr_learn_q(int rows, int cols, const float* d_values, const uint8_t* d_sample_mask, const mpr_params* h_params,
                       const float* h_q, int n_q, double holdout_fraction, void* d_workspace, size_t workspace_bytes,
                       void* cuda_stream, float* h_q_hat, double* h_scores, double* h_T)
{
    LearnLayout L;
    if (!d_values || !d_sample_mask || !h_params || !h_q || n_q < 1 || !h_q_hat || !h_scores ||
        !(holdout_fraction > 0.0 && holdout_fraction < 1.0) || h_params->struct_size != sizeof(mpr_params) ||
        !learn_layout(rows, cols, &L)) return MPR_ERR_ARG;
    for (int k = 0; k < n_q; ++k)
        if (!(h_q[k] > 0.0f && h_q[k] <= 0.5f)) return MPR_ERR_ARG;
    if (!d_workspace || workspace_bytes < L.total || ((uintptr_t)d_workspace & 255u)) return MPR_ERR_WORKSPACE;
    char* base = (char*)d_workspace;
    uint8_t* train = (uint8_t*)(base + L.train); uint8_t* held = (uint8_t*)(base + L.held);
    float* pred = (float*)(base + L.pred);
    double* partials = (double*)(base + L.partials);
    unsigned long long* count = (unsigned long long*)(base + L.count);
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const uint32_t N = (uint32_t)((size_t)rows * cols);
    PhiloxKeys keys;
    for (int r = 0; r < PHILOX_ROUNDS; ++r) {
        keys.rk0[r] = (uint32_t)h_params->seed + (uint32_t)r * 0x9E3779B9u;
        keys.rk1[r] = (uint32_t)(h_params->seed >> 32) + (uint32_t)r * 0xBB67AE85u;
    }
    k_holdout<<<cdiv(N, 256), 256, 0, st>>>(keys, d_sample_mask, train, held, N, 0u, (float)holdout_fraction);
    if (!cuda_ok(cudaGetLastError(), "k_holdout")) return MPR_ERR_CUDA;
    mpr_ctx* ctx = nullptr;
    mpr_status s = mpr_create(&ctx, 1, rows, cols, d_values, train, base + L.ctx, L.ctx == 0 ? L.train : L.train - L.ctx, cuda_stream);
    if (s != MPR_OK) return s;
    int best = -1;
    for (int k = 0; k < n_q && s == MPR_OK; ++k) {
        // T of this candidate: the remaining samples' specific energy at this q (Eq. 4) through the equipartition line
        double e_s = 0.0; uint64_t pairs = 0;
        const float one = 1.0f; float T = 0.0f;
        ctx->d.q = h_q[k];
        s = mpr_sample_energy(ctx, &e_s, &pairs);
        if (s == MPR_OK && pairs == 0) s = MPR_ERR_NO_SAMPLES;
        if (s == MPR_OK) s = mpr_default_ladder(rows, cols, e_s, &one, 1, &T);
        mpr_params prm = *h_params;
        prm.q = h_q[k];
        if (s == MPR_OK) s = mpr_set_params(ctx, &prm, &T);
        if (s == MPR_OK) s = mpr_equilibrate(ctx);
        if (s == MPR_OK) s = mpr_simulate(ctx);
        if (s == MPR_OK) s = mpr_predict(ctx, pred);
        if (s != MPR_OK) break;
        if (!cuda_ok(cudaMemsetAsync(count, 0, sizeof *count, st), "memset")) { s = MPR_ERR_CUDA; break; }
        k_cv_error<<<ENERGY_BLOCKS, ENERGY_THREADS, 0, st>>>(d_values, pred, held, N, partials, count);
        k_cv_finish<<<1, 32, 0, st>>>(partials, ENERGY_BLOCKS);
        double sum = 0.0; unsigned long long n_held = 0;
        if (!cuda_ok(cudaMemcpyAsync(&sum, partials, sizeof sum, cudaMemcpyDeviceToHost, st), "copy") ||
            !cuda_ok(cudaMemcpyAsync(&n_held, count, sizeof n_held, cudaMemcpyDeviceToHost, st), "copy") ||
            !cuda_ok(cudaStreamSynchronize(st), "sync")) { s = MPR_ERR_CUDA; break; }
        if (n_held == 0) { s = MPR_ERR_NO_SAMPLES; break; }          // nothing was withheld: no score
        h_scores[k] = std::sqrt(sum / (double)n_held);
        if (h_T) h_T[k] = (double)T;
        if (best < 0 || h_scores[k] < h_scores[best]) best = k;
    }
    mpr_destroy(ctx);
    if (s != MPR_OK) return s;
    *h_q_hat = h_q[best];
    return MPR_OK;
}

mpr_status mpr_get_angles(mpr_ctx* ctx, float* d_phi)
{
    if (!ctx || !d_phi) return MPR_ERR_ARG;
    ENTER(ctx);
    if (ctx->state != READY) return MPR_ERR_STATE;
    const Dev& d = ctx->d;
    if (ctx->dirty) {        // otherwise d.phi already holds the state exactly (initial draw or import)
        k_export_angles<<<site_grid(ctx), 256, 0, ctx->stream>>>(d);
        CU_LAUNCH();
        ctx->dirty = false;
    }
    CU(cudaMemcpyAsync(d_phi, d.phi, sizeof(float) * (size_t)d.N * d.batch, cudaMemcpyDeviceToDevice, ctx->stream));
    return MPR_OK;
}

mpr_status mpr_set_angles(mpr_ctx* ctx, const float* d_phi)
{
    if (!ctx || !d_phi) return MPR_ERR_ARG;
    ENTER(ctx);
    if (ctx->state != READY) return MPR_ERR_STATE;
    k_import_angles<<<site_grid(ctx), 256, 0, ctx->stream>>>(ctx->d, d_phi);
    CU_LAUNCH();
    ctx->dirty = false;
    ctx->forked = false;
    if (ctx->slab) return halo_exchange(ctx, ctx->cur);       // the ghost rows are the neighbours' own rows, whatever d_phi held there
    return MPR_OK;
}

mpr_status mpr_set_sweep_index(mpr_ctx* ctx, uint32_t t)
{
    if (!ctx) return MPR_ERR_ARG;
    ENTER(ctx);
    if (ctx->state != READY) return MPR_ERR_STATE;
    k_set_t<<<cdiv(ctx->d.batch, 128), 128, 0, ctx->stream>>>(ctx->d, t);
    CU_LAUNCH();
    ctx->forked = false;
    return MPR_OK;
}

mpr_status mpr_sweep(mpr_ctx* ctx, uint32_t n_sweeps, double a, uint64_t* h_accepted)
{
    if (!ctx || !(a >= 1.0) || !std::isfinite(a)) return MPR_ERR_ARG;
    ENTER(ctx);
    if (ctx->state != READY) return MPR_ERR_STATE;
    const Dev& d = ctx->d;
    k_set_a<<<cdiv(d.nv, 128), 128, 0, ctx->stream>>>(d, 0, a, 1);       // also zeroes the accepted counters
    CU_LAUNCH();
    note_a(ctx, a);
    ctx->forked = false;
    uint32_t t_off = 0, flip = 0;
    mpr_status rs = launch_sweeps(ctx, n_sweeps, &t_off, &flip, h_accepted ? PASS_COUNT : 0u, 0);
    if (rs != MPR_OK) return rs;
    k_commit<<<cdiv(d.batch, 128), 128, 0, ctx->stream>>>(d, 0, d.batch, t_off, flip, 0);
    CU_LAUNCH();
    ctx->cur ^= flip;
    if (h_accepted) {
        mpr_status s = fetch_states(ctx);
        if (s != MPR_OK) return s;
        for (int b = 0; b < d.batch; ++b) h_accepted[b] = ctx->h_states[b].accepted;
    }
    return MPR_OK;
}

mpr_status mpr_energy(mpr_ctx* ctx, double* h_e)
{
    if (!ctx || !h_e) return MPR_ERR_ARG;
    ENTER(ctx);
    if (ctx->state != READY) return MPR_ERR_STATE;
    mpr_status s = launch_energy(ctx);
    if (s != MPR_OK) return s;
    if (ctx->slab) {        // this slab's share (own rows), summed over the slabs, over the bonds of the whole grid
        k_slab_partial<<<1, REDUCE_THREADS, 0, ctx->stream>>>(ctx->d, ctx->energy_blocks);
        CU_LAUNCH();
        s = fetch_states(ctx);
        if (s != MPR_OK) return s;
        double H = ctx->h_states[0].e_query;
        if (ctx->slab_cfg.allreduce(ctx->slab_cfg.user, &H, 1, MPR_REDUCE_SUM)) return MPR_ERR_COMM;
        h_e[0] = H / ctx->d.n_bonds;
        return MPR_OK;
    }
    k_energy_query<<<ctx->d.batch, REDUCE_THREADS, 0, ctx->stream>>>(ctx->d, ctx->energy_blocks);
    CU_LAUNCH();
    s = fetch_states(ctx);
    if (s != MPR_OK) return s;
    for (int b = 0; b < ctx->d.batch; ++b) h_e[b] = ctx->h_states[b].e_query;
    return MPR_OK;
}

mpr_status mpr_get_transform(mpr_ctx* ctx, float* h_zmin, float* h_zmax)
{
    if (!ctx || !h_zmin || !h_zmax) return MPR_ERR_ARG;
    for (int b = 0; b < ctx->d.batch; ++b) { h_zmin[b] = ctx->h_states[b].zmin; h_zmax[b] = ctx->h_states[b].zmax; }
    return MPR_OK;      // z_min / z_max never change after mpr_create, which fetched them
}

mpr_status mpr_get_mask_bits(mpr_ctx* ctx, uint32_t* d_bits)
{
    if (!ctx || !d_bits) return MPR_ERR_ARG;
    ENTER(ctx);
    CU(cudaMemcpyAsync(d_bits, ctx->d.bits, sizeof(uint32_t) * (size_t)ctx->d.words * ctx->d.batch,
                       cudaMemcpyDeviceToDevice, ctx->stream));
    return MPR_OK;
}

mpr_status mpr_get_stats(mpr_ctx* ctx, mpr_stats* h_out)
{
    if (!ctx || !h_out) return MPR_ERR_ARG;
    ENTER(ctx);
    mpr_status s = fetch_states(ctx);
    if (s != MPR_OK) return s;
    for (int b = 0; b < ctx->d.batch; ++b) {
        const GridState& g = ctx->h_states[b];
        mpr_stats& o = h_out[b];
        o.equil_sweeps = g.i; o.t = g.t; o.equilibrated = g.done;
        o.realizations = 0;            // pooled over the grid's chains
        for (int c = 0; c < ctx->d.chains; ++c) o.realizations += ctx->h_states[b + c * ctx->d.batch].realizations;
        o.n_free = (uint64_t)g.n_free[0] + g.n_free[1];
        o.n_samples = g.n_samples;
        o.n_bonds = (uint64_t)ctx->d.n_bonds;
        o.a = g.a; o.k = g.k; o.A_last = g.A_last; o.e_last = g.e_last;
        o.z_min = g.zmin; o.z_max = g.zmax;
    }
    return MPR_OK;
}

mpr_status mpr_get_launch_count(mpr_ctx* ctx, uint64_t* h_count)
{
    if (!ctx || !h_count) return MPR_ERR_ARG;
    *h_count = ctx->launches;
    return MPR_OK;
}

mpr_status mpr_set_pass_depth(mpr_ctx* ctx, uint32_t k)
{
    if (!ctx) return MPR_ERR_ARG;
    uint32_t most = ctx->d.ntiles == 1 ? 1024u : (uint32_t)(ctx->d.H / 2);
    if (ctx->slab && most > (uint32_t)(SLAB_GHOST / 2)) most = SLAB_GHOST / 2;
    if (k > most) return MPR_ERR_ARG;
    ctx->k_max = k ? k : most;
    return MPR_OK;
}

mpr_status mpr_set_grid_group(mpr_ctx* ctx, int grids)
{
    if (!ctx || grids < 0) return MPR_ERR_ARG;
    ctx->group = grids;
    return MPR_OK;
}

mpr_status mpr_get_tiling(mpr_ctx* ctx, int* h_tile_rows, int* h_tile_cols, int* h_halo, uint32_t* h_pass_depth)
{
    if (!ctx || !h_tile_rows || !h_tile_cols || !h_halo || !h_pass_depth) return MPR_ERR_ARG;
    *h_tile_rows = ctx->d.TR; *h_tile_cols = ctx->d.TC; *h_halo = ctx->d.H; *h_pass_depth = ctx->k_max;
    return MPR_OK;
}

}  // extern "C"

#include "mpr_f64_api.inl"
#include "mpr_noalloc.inl"
