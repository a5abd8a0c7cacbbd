// mpr_f64_api.inl -- host controller and C ABI (include/mpr.h, "double-precision path") of the kernels in
// mpr_f64.cuh.  Included at the end of mpr_api.cu (uses its CU / cuda_ok / align_up / cdiv helpers).

namespace {

struct Layout64 { size_t state, done, partials, values, phi, bits, list, list_counts, vec, acc, acc2, tstate, tile_meta, entries, total; };

// tiles of the double-precision tile pass: 64 x 64 cores with a halo of 8 (4 sweeps per pass), lower cores of the same
// pitch when 64 rows would not give every SM its two CTAs; lists by the fp32 path's kernels (frame offsets, pitch FC)
void choose_tiles64(int rows, int cols, Geometry* g)
{
    int TR = 64;
    const long ntx = (cols + 63) / 64;
    if (ntx * ((rows + 63) / 64) < 148L * 2L)
        for (int tr = 16; tr < 64; tr += 8)
            if (ntx * ((rows + tr - 1) / tr) <= 148L * 2L) { TR = tr; break; }
    g->TR = TR; g->TC = 64; g->H = 8; g->FR = TR + 16;
    g->FC = ((64 + 16 + 1) & ~3) + 2;
    g->ntx = (int)ntx; g->nty = (rows + TR - 1) / TR; g->ntiles = g->ntx * g->nty;
    g->entry_stride = (size_t)g->ntiles * (((size_t)g->FR * g->FC + 31) & ~(size_t)15);
}

bool geometry64(int rows, int cols, uint32_t* N, uint32_t* words)
{
    if (rows < 2 || cols < 2 || rows > 65534 || cols > 65534) return false;
    const uint64_t n = (uint64_t)rows * (uint64_t)cols;
    if (n >= (1ull << 31)) return false;
    *N = (uint32_t)n; *words = (uint32_t)((n + 31) / 32);
    return true;
}

Layout64 make_layout64(int rows, int cols, uint32_t N, uint32_t words)
{
    Layout64 L;
    Geometry g;
    choose_tiles64(rows, cols, &g);
    size_t o = 0;
    auto take = [&](size_t bytes) { size_t at = o; o = align_up(o + bytes); return at; };
    L.state    = take(sizeof(mpr64::State64));
    L.done     = take(sizeof(uint32_t));
    L.partials = take(sizeof(double) * 4 * mpr64::MM_BLOCKS);
    L.values   = take(sizeof(double) * N);
    L.phi      = take(sizeof(double) * N);
    L.bits     = take(sizeof(uint32_t) * words);
    L.list     = take(sizeof(uint32_t) * N);
    L.list_counts = take(sizeof(uint32_t) * 2 * cdiv(words, mpr64::LIST_THREADS));
    L.vec      = take(sizeof(double2) * 2 * 2 * (size_t)rows * (size_t)((cols + 1) / 2));       // two buffers of two planes
    L.acc      = take(sizeof(double) * N);
    L.acc2     = take(sizeof(double) * N);
    L.tstate   = take(sizeof(GridState));
    L.tile_meta = take(sizeof(TileMeta) * (size_t)g.ntiles);
    L.entries  = take(sizeof(uint16_t) * (g.entry_stride + 16));
    L.total = o;
    return L;
}

}  // namespace

struct mpr64_ctx {
    mpr64::Dev64   d;
    cudaStream_t   stream;
    mpr_params     prm;
    RunState       state;
    int            device, energy_blocks;
    uint32_t       n_colour[2];   // prediction sites per colour (lengths of the site lists)
    uint64_t       launches;
    uint32_t       h_done;        // host copy of the done flag
    mpr64::State64 h_state;
    bool           qhalf, dirty;
    uint64_t       n_realizations;   // realizations accumulated since mpr64_set_params
    // the tile pass (k64_tilepass): tiling and lists in the fp32 path's format, TMA descriptors [buffer][plane]
    mpr::Dev       dt;
    alignas(64) CUtensorMap map[2][2];
    double2*       vec_buf[2];
    uint32_t       cur;              // d.vec = vec_buf[cur]
    size_t         tile_smem;
    uint32_t       k_max;
};

namespace {

#define ENTER64(ctx) do { if (!cuda_ok(cudaSetDevice((ctx)->device), "cudaSetDevice")) return MPR_ERR_CUDA; } while (0)

mpr_status fetch_state64(mpr64_ctx* ctx)
{
    CU(cudaMemcpyAsync(&ctx->h_state, ctx->d.state, sizeof(mpr64::State64), cudaMemcpyDeviceToHost, ctx->stream));
    CU(cudaStreamSynchronize(ctx->stream));
    return MPR_OK;
}

typedef void (*half_kernel)(mpr64::Dev64, const uint32_t*, uint32_t, uint32_t, int, int);
typedef void (*tile_kernel64)(const CUtensorMap, const CUtensorMap, const mpr64::Dev64, const mpr::Dev, double2*, uint32_t, uint32_t);
tile_kernel64 pick_tile_kernel64(bool qhalf, int or_mode)
{
    using namespace mpr64;
    if (qhalf) return or_mode == 0 ? k64_tilepass<true, 0> : or_mode == 1 ? k64_tilepass<true, 1> : k64_tilepass<true, 2>;
    return or_mode == 0 ? k64_tilepass<false, 0> : k64_tilepass<false, 2>;
}

void set_cur64(mpr64_ctx* ctx, uint32_t cur)
{
    ctx->cur = cur;
    ctx->d.vec = ctx->vec_buf[cur]; ctx->d.vec_other = ctx->vec_buf[cur ^ 1u];
}

// n sweeps without the accepted count, as tile passes of up to k_max sweeps (sweep indices state.t + *t_off ...)
mpr_status launch_passes64(mpr64_ctx* ctx, uint32_t n, uint32_t* t_off)
{
    const tile_kernel64 kern = pick_tile_kernel64(ctx->qhalf, (int)ctx->prm.or_mode);
    while (n) {
        const uint32_t K = n < ctx->k_max ? n : ctx->k_max;
        kern<<<ctx->dt.ntiles, mpr64::T64_THREADS, ctx->tile_smem, ctx->stream>>>(ctx->map[ctx->cur][0], ctx->map[ctx->cur][1], ctx->d,
                                                                                   ctx->dt, ctx->d.vec_other, K, *t_off);
        CU_LAUNCH();
        set_cur64(ctx, ctx->cur ^ 1u);
        *t_off += K; n -= K;
    }
    ctx->dirty = true;
    return MPR_OK;
}

// TMA descriptor of one colour plane of one vector buffer: [rows][2 * half] eight-byte words (a double2 is two), box =
// one tile frame's share of the plane; out-of-grid elements arrive as zeros (open boundary, L109)
mpr_status make_plane_map64(mpr64_ctx* ctx, int buf, int plane)
{
    void* fn = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (!cuda_ok(cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres), "cudaGetDriverEntryPoint") ||
        qres != cudaDriverEntryPointSuccess || !fn) return MPR_ERR_CUDA;
    const mpr64::Dev64& d = ctx->d;
    const cuuint64_t dims[2] = {(cuuint64_t)d.half * 2u, (cuuint64_t)d.rows};
    const cuuint64_t strides[1] = {(cuuint64_t)d.half * sizeof(double2)};
    const cuuint32_t box[2] = {(cuuint32_t)ctx->dt.FC, (cuuint32_t)ctx->dt.FR};          // FC / 2 double2 = FC words
    const cuuint32_t estr[2] = {1u, 1u};
    const CUresult r = ((PFN_cuTensorMapEncodeTiled)fn)(&ctx->map[buf][plane], CU_TENSOR_MAP_DATA_TYPE_UINT64, 2,
                                                         (void*)(ctx->vec_buf[buf] + (size_t)plane * d.plane), dims, strides, box, estr,
                                                         CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                                                         CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) {
        snprintf(g_cuda_err, sizeof g_cuda_err, "cuTensorMapEncodeTiled (double planes) failed with CUresult %d", (int)r);
        return MPR_ERR_CUDA;
    }
    return MPR_OK;
}
half_kernel pick_half_kernel(bool qhalf, int or_mode)
{
    using namespace mpr64;
    if (qhalf) return or_mode == 0 ? k64_halfsweep<true, 0> : or_mode == 1 ? k64_halfsweep<true, 1> : k64_halfsweep<true, 2>;
    return or_mode == 0 ? k64_halfsweep<false, 0> : k64_halfsweep<false, 2>;
}

// one sweep at sweep index state.t + t_off: colour 0 (the one holding the upper-left node), then colour 1 (L261-265)
// check_done: the sweep does nothing once the equilibration has stopped (State64::done)
mpr_status launch_sweep64(mpr64_ctx* ctx, uint32_t t_off, int count, int check_done = 0)
{
    const half_kernel kern = pick_half_kernel(ctx->qhalf, (int)ctx->prm.or_mode);
    const uint32_t* sites = ctx->d.list;
    for (int colour = 0; colour < 2; ++colour) {
        if (ctx->n_colour[colour]) {
            kern<<<cdiv(ctx->n_colour[colour], 256), 256, 0, ctx->stream>>>(ctx->d, sites, ctx->n_colour[colour], t_off, count, check_done);
            CU_LAUNCH();
        }
        sites += ctx->n_colour[colour];
    }
    ctx->dirty = true;
    return MPR_OK;
}

}  // namespace

extern "C" {

mpr_status mpr64_query_workspace(int rows, int cols, size_t* bytes)
{
    uint32_t N, words;
    if (!bytes || !geometry64(rows, cols, &N, &words)) return MPR_ERR_ARG;
    *bytes = make_layout64(rows, cols, N, words).total;
    return MPR_OK;
}

mpr_status mpr64_destroy(mpr64_ctx* ctx)
{
    if (!ctx) return MPR_ERR_ARG;
    delete ctx;
    return MPR_OK;
}

mpr_status mpr64_create(mpr64_ctx** out, int rows, int cols, const double* d_values, const uint8_t* d_sample_mask,
                        void* d_workspace, size_t workspace_bytes, void* cuda_stream)
{
    uint32_t N, words;
    if (!out || !d_values || !d_sample_mask || !geometry64(rows, cols, &N, &words)) return MPR_ERR_ARG;
    const Layout64 lay = make_layout64(rows, cols, N, words);
    if (!d_workspace || workspace_bytes < lay.total || ((uintptr_t)d_workspace & 255u)) return MPR_ERR_WORKSPACE;
    mpr64_ctx* ctx = new (std::nothrow) mpr64_ctx();
    if (!ctx) return MPR_ERR_ARG;
    memset(ctx, 0, sizeof *ctx);
    ctx->stream = (cudaStream_t)cuda_stream;
    {
        cudaPointerAttributes attr;
        if (!cuda_ok(cudaPointerGetAttributes(&attr, d_workspace), "cudaPointerGetAttributes") ||
            attr.type != cudaMemoryTypeDevice) { delete ctx; return MPR_ERR_WORKSPACE; }
        ctx->device = attr.device;
        if (!cuda_ok(cudaSetDevice(ctx->device), "cudaSetDevice")) { delete ctx; return MPR_ERR_CUDA; }
    }
    ctx->state = CREATED;
    char* base = (char*)d_workspace;
    mpr64::Dev64& d = ctx->d;
    d.state = (mpr64::State64*)(base + lay.state);
    d.done_flag = (uint32_t*)(base + lay.done);
    d.partials = (double*)(base + lay.partials);
    d.values = (double*)(base + lay.values);
    d.phi = (double*)(base + lay.phi);
    d.bits = (uint32_t*)(base + lay.bits);
    d.list = (uint32_t*)(base + lay.list);
    d.list_counts = (uint32_t*)(base + lay.list_counts);
    d.list_blocks = cdiv(words, mpr64::LIST_THREADS);
    ctx->vec_buf[0] = (double2*)(base + lay.vec);
    ctx->vec_buf[1] = ctx->vec_buf[0] + 2 * (size_t)rows * (size_t)((cols + 1) / 2);
    set_cur64(ctx, 0);
    d.acc = (double*)(base + lay.acc);
    d.acc2 = (double*)(base + lay.acc2);
    d.rows = rows; d.cols = cols; d.N = N; d.words = words;
    d.half = (cols + 1) / 2; d.plane = (uint32_t)rows * (uint32_t)d.half;
    d.q = 0.5; d.inv_q = 2.0;
    d.n_bonds = (double)rows * (cols - 1) + (double)cols * (rows - 1);
    ctx->energy_blocks = rows < mpr64::E_BLOCKS ? rows : mpr64::E_BLOCKS;
    auto fail = [&](mpr_status s) { mpr64_destroy(ctx); return s; };
    unsigned mm_blocks = cdiv(N, 256 * 8);
    if (mm_blocks > (unsigned)mpr64::MM_BLOCKS) mm_blocks = mpr64::MM_BLOCKS;
    mpr64::k64_minmax<<<mm_blocks, 256, 0, ctx->stream>>>(d, d_values, d_sample_mask);
    mpr64::k64_minmax_finish<<<1, 1, 0, ctx->stream>>>(d, (int)mm_blocks);
    mpr64::k64_transform<<<cdiv((size_t)words * 32, 256), 256, 0, ctx->stream>>>(d, d_values, d_sample_mask);
    mpr64::k64_list_count<<<d.list_blocks, mpr64::LIST_THREADS, 0, ctx->stream>>>(d);
    mpr64::k64_list_scan<<<1, 1, 0, ctx->stream>>>(d);
    mpr64::k64_list_fill<<<d.list_blocks, mpr64::LIST_THREADS, 0, ctx->stream>>>(d);
    ctx->launches += 6;
    if (!cuda_ok(cudaGetLastError(), "create kernels")) return fail(MPR_ERR_CUDA);
    mpr_status st = fetch_state64(ctx);
    if (st != MPR_OK) return fail(st);
    const uint32_t e = ctx->h_state.err_flags;
    if (e & mpr::ERRF_NO_SAMPLES) return fail(MPR_ERR_NO_SAMPLES);
    if (e & mpr::ERRF_NONFINITE) return fail(MPR_ERR_NONFINITE);
    if (e & mpr::ERRF_DEGENERATE) return fail(MPR_ERR_DEGENERATE_RANGE);
    if (e & mpr::ERRF_NO_FREE) return fail(MPR_ERR_NO_FREE);
    ctx->n_colour[0] = ctx->h_state.n_colour[0]; ctx->n_colour[1] = ctx->h_state.n_colour[1];
    // the tile pass: tiles and per-tile entry lists in the fp32 path's format, built by its kernels on this grid's bitmask
    {
        Geometry g;
        choose_tiles64(rows, cols, &g);
        mpr::Dev& t = ctx->dt;
        memset(&t, 0, sizeof t);
        t.states = (GridState*)(base + lay.tstate);
        t.bits = d.bits; t.tile_meta = (TileMeta*)(base + lay.tile_meta); t.entries = (uint16_t*)(base + lay.entries);
        t.batch = 1; t.rows = rows; t.cols = cols; t.chains = 1; t.nv = 1;
        t.N = N; t.words = words;
        t.entry_stride = g.entry_stride; t.tile_entries = (uint32_t)(g.entry_stride / (size_t)g.ntiles);
        t.TR = g.TR; t.TC = g.TC; t.H = g.H; t.FR = g.FR; t.FC = g.FC; t.ntx = g.ntx; t.nty = g.nty; t.ntiles = g.ntiles;
        t.fc_inv = (uint32_t)(((1u << 24) + (uint32_t)g.FC - 1u) / (uint32_t)g.FC);
        t.own_r0 = 0; t.own_r1 = rows;
        // the pads of an odd-width grid's planes stay zero (the frame loads read them as neighbours)
        if (!cuda_ok(cudaMemsetAsync(ctx->vec_buf[0], 0, sizeof(double2) * 4 * (size_t)rows * (size_t)d.half, ctx->stream), "memset vec")) return fail(MPR_ERR_CUDA);
        k_tile_count<<<dim3(g.ntiles, 1), 256, 0, ctx->stream>>>(t);
        k_tile_scan<<<1, 32, 0, ctx->stream>>>(t);
        const size_t fill_smem = (size_t)g.FR * g.FC * sizeof(uint16_t);
        k_tile_fill<<<dim3(g.ntiles, 1), 256, fill_smem, ctx->stream>>>(t);       // <= 80 x 82 x 2 bytes: below the default limit
        ctx->launches += 3;
        GridState hs;
        if (!cuda_ok(cudaMemcpyAsync(&hs, t.states, sizeof hs, cudaMemcpyDeviceToHost, ctx->stream), "copy") ||
            !cuda_ok(cudaStreamSynchronize(ctx->stream), "sync") || !cuda_ok(cudaGetLastError(), "tile lists")) return fail(MPR_ERR_CUDA);
        t.max_entries = (hs.max_tile_entries + 15u) & ~15u;
        ctx->tile_smem = (size_t)2 * g.FR * (g.FC / 2) * sizeof(double2) + (size_t)t.max_entries * sizeof(uint16_t);
        ctx->k_max = (uint32_t)(g.H / 2);
        for (int qh = 0; qh < 2; ++qh)
            for (int om = 0; om < 3; ++om) {
                if (!qh && om == 1) continue;
                if (!cuda_ok(cudaFuncSetAttribute((const void*)pick_tile_kernel64(qh, om), cudaFuncAttributeMaxDynamicSharedMemorySize,
                                                  (int)ctx->tile_smem), "cudaFuncSetAttribute")) return fail(MPR_ERR_CUDA);
            }
        for (int b = 0; b < 2; ++b)
            for (int p = 0; p < 2; ++p) { st = make_plane_map64(ctx, b, p); if (st != MPR_OK) return fail(st); }
    }
    *out = ctx;
    return MPR_OK;
}

mpr_status mpr64_set_params(mpr64_ctx* ctx, const mpr_params* p, double T)
{
    if (!ctx || !p || p->struct_size != sizeof(mpr_params)) return MPR_ERR_ARG;
    ENTER64(ctx);
    if (!(p->q > 0.0f && p->q <= 0.5f) || p->M < 1 || p->sweeps_per_real < 1 || p->n_f < 1 ||
        p->n_fit < 2 || p->n_fit > (uint32_t)mpr::MAX_NFIT || !(p->k_a > 0.0f) || !std::isfinite(p->A_targ) ||
        p->or_mode > 2 || p->a_eq_mode > 1 || !(T > 0.0) || !std::isfinite(T))
        return MPR_ERR_ARG;
    if (p->or_mode == 1 && p->q != 0.5f) return MPR_ERR_UNSUPPORTED;
    ctx->prm = *p;
    ctx->qhalf = p->q == 0.5f;
    mpr64::Dev64& d = ctx->d;
    for (int r = 0; r < mpr::PHILOX_ROUNDS; ++r) {
        d.rk0[r] = (uint32_t)p->seed + (uint32_t)r * 0x9E3779B9u;
        d.rk1[r] = (uint32_t)(p->seed >> 32) + (uint32_t)r * 0xBB67AE85u;
    }
    d.q = (double)p->q; d.inv_q = 1.0 / (double)p->q;
    d.bc = cos(d.q * mpr64::TWO_PI_D); d.bs = sin(d.q * mpr64::TWO_PI_D);
    d.n_f = p->n_f; d.n_fit = p->n_fit; d.equil_cap = p->equil_cap;
    d.A_targ = (double)p->A_targ; d.k_a = (double)p->k_a;
    mpr64::k64_edit<<<1, 1, 0, ctx->stream>>>(d, 0, T, 0u, 0u);
    CU_LAUNCH();
    CU(cudaMemsetAsync(d.acc, 0, sizeof(double) * d.N, ctx->stream));
    CU(cudaMemsetAsync(d.acc2, 0, sizeof(double) * d.N, ctx->stream));
    mpr64::k64_init_state<<<cdiv(d.N, 256), 256, 0, ctx->stream>>>(d);
    CU_LAUNCH();
    ctx->state = READY;
    ctx->dirty = false;
    ctx->n_realizations = 0;
    return MPR_OK;
}

mpr_status mpr64_equilibrate(mpr64_ctx* ctx)
{
    if (!ctx) return MPR_ERR_ARG;
    ENTER64(ctx);
    if (ctx->state != READY) return MPR_ERR_STATE;
    const mpr64::Dev64& d = ctx->d;
    const uint32_t cap = ctx->prm.equil_cap;
    // The controller checks the slope after the sweep with index i when i >= n_fit and i % n_f == 0 (step 5.4), so the
    // run can only stop after i + 1 sweeps with i such an index: the host polls the flag exactly there (and a sweep
    // enqueued after the stop does nothing: check_done).
    const uint32_t n_f = ctx->prm.n_f;
    uint32_t issued = 0, chunk = (ctx->prm.n_fit + n_f - 1) / n_f * n_f + 1;
    while (issued < cap) {
        if (chunk > cap - issued) chunk = cap - issued;
        for (uint32_t j = 0; j < chunk; ++j) {
            mpr_status s = launch_sweep64(ctx, 0, 1, 1);    // 5.1, accepted proposals counted
            if (s != MPR_OK) return s;
            mpr64::k64_energy<<<ctx->energy_blocks, mpr64::E_THREADS, 0, ctx->stream>>>(d);      // 5.3
            CU_LAUNCH();
            mpr64::k64_controller<<<1, 32, 0, ctx->stream>>>(d, ctx->energy_blocks);             // 5.2, 5.4, 5.5
            CU_LAUNCH();
        }
        issued += chunk;
        CU(cudaMemcpyAsync(&ctx->h_done, d.done_flag, sizeof(uint32_t), cudaMemcpyDeviceToHost, ctx->stream));
        CU(cudaStreamSynchronize(ctx->stream));
        if (ctx->h_done) break;
        chunk = n_f;
    }
    return MPR_OK;
}

mpr_status mpr64_simulate(mpr64_ctx* ctx)
{
    if (!ctx) return MPR_ERR_ARG;
    ENTER64(ctx);
    if (ctx->state != READY) return MPR_ERR_STATE;
    const mpr64::Dev64& d = ctx->d;
    if (ctx->prm.a_eq_mode == 1) { mpr64::k64_edit<<<1, 1, 0, ctx->stream>>>(d, 1, 1.0, 0u, 0u); CU_LAUNCH(); }
    uint32_t t_off = 0;
    for (uint32_t j = 0; j < ctx->prm.M; ++j) {
        mpr_status s = launch_passes64(ctx, ctx->prm.sweeps_per_real, &t_off);        // tile passes of up to 4 sweeps
        if (s != MPR_OK) return s;
        mpr64::k64_accumulate<<<cdiv(ctx->d.N, 256), 256, 0, ctx->stream>>>(ctx->d);    // step 6.3
        CU_LAUNCH();
    }
    mpr64::k64_edit<<<1, 1, 0, ctx->stream>>>(d, 2, 0.0, t_off, ctx->prm.M);
    CU_LAUNCH();
    ctx->n_realizations += ctx->prm.M;
    return MPR_OK;
}

mpr_status mpr64_predict(mpr64_ctx* ctx, double* d_out)
{
    if (!ctx || !d_out) return MPR_ERR_ARG;
    ENTER64(ctx);
    if (ctx->state != READY || ctx->n_realizations == 0) return MPR_ERR_STATE;     // the mean of no realization is 0 / 0
    mpr64::k64_predict<<<cdiv(ctx->d.N, 256), 256, 0, ctx->stream>>>(ctx->d, d_out, 0);
    CU_LAUNCH();
    return MPR_OK;
}

mpr_status mpr64_predict_std(mpr64_ctx* ctx, double* d_out)
{
    if (!ctx || !d_out) return MPR_ERR_ARG;
    ENTER64(ctx);
    if (ctx->state != READY) return MPR_ERR_STATE;
    mpr_status s = fetch_state64(ctx);
    if (s != MPR_OK) return s;
    if (ctx->h_state.realizations < 2u) return MPR_ERR_STATE;
    mpr64::k64_predict<<<cdiv(ctx->d.N, 256), 256, 0, ctx->stream>>>(ctx->d, d_out, 1);
    CU_LAUNCH();
    return MPR_OK;
}

mpr_status mpr64_get_angles(mpr64_ctx* ctx, double* d_phi)
{
    if (!ctx || !d_phi) return MPR_ERR_ARG;
    ENTER64(ctx);
    if (ctx->state != READY) return MPR_ERR_STATE;
    if (ctx->dirty) {
        mpr64::k64_export_angles<<<cdiv(ctx->d.N, 256), 256, 0, ctx->stream>>>(ctx->d);
        CU_LAUNCH();
        ctx->dirty = false;
    }
    CU(cudaMemcpyAsync(d_phi, ctx->d.phi, sizeof(double) * ctx->d.N, cudaMemcpyDeviceToDevice, ctx->stream));
    return MPR_OK;
}

mpr_status mpr64_set_angles(mpr64_ctx* ctx, const double* d_phi)
{
    if (!ctx || !d_phi) return MPR_ERR_ARG;
    ENTER64(ctx);
    if (ctx->state != READY) return MPR_ERR_STATE;
    mpr64::k64_import_angles<<<cdiv(ctx->d.N, 256), 256, 0, ctx->stream>>>(ctx->d, d_phi);
    CU_LAUNCH();
    ctx->dirty = false;
    return MPR_OK;
}

mpr_status mpr64_set_sweep_index(mpr64_ctx* ctx, uint32_t t)
{
    if (!ctx) return MPR_ERR_ARG;
    ENTER64(ctx);
    if (ctx->state != READY) return MPR_ERR_STATE;
    mpr64::k64_edit<<<1, 1, 0, ctx->stream>>>(ctx->d, 3, 0.0, t, 0u);
    CU_LAUNCH();
    return MPR_OK;
}

mpr_status mpr64_sweep(mpr64_ctx* ctx, uint32_t n_sweeps, double a, uint64_t* h_accepted)
{
    if (!ctx || !(a >= 1.0) || !std::isfinite(a)) return MPR_ERR_ARG;
    ENTER64(ctx);
    if (ctx->state != READY) return MPR_ERR_STATE;
    mpr64::k64_edit<<<1, 1, 0, ctx->stream>>>(ctx->d, 1, a, 0u, 0u);        // also zeroes the accepted counter
    CU_LAUNCH();
    if (h_accepted) {
        for (uint32_t w = 0; w < n_sweeps; ++w) {
            mpr_status s = launch_sweep64(ctx, w, 1);
            if (s != MPR_OK) return s;
        }
    } else {
        uint32_t t_off = 0;
        mpr_status s = launch_passes64(ctx, n_sweeps, &t_off);
        if (s != MPR_OK) return s;
    }
    mpr64::k64_edit<<<1, 1, 0, ctx->stream>>>(ctx->d, 2, 0.0, n_sweeps, 0u);
    CU_LAUNCH();
    if (h_accepted) {
        mpr_status s = fetch_state64(ctx);
        if (s != MPR_OK) return s;
        *h_accepted = ctx->h_state.accepted;
    }
    return MPR_OK;
}

mpr_status mpr64_energy(mpr64_ctx* ctx, double* h_e)
{
    if (!ctx || !h_e) return MPR_ERR_ARG;
    ENTER64(ctx);
    if (ctx->state != READY) return MPR_ERR_STATE;
    mpr64::k64_energy<<<ctx->energy_blocks, mpr64::E_THREADS, 0, ctx->stream>>>(ctx->d);
    CU_LAUNCH();
    mpr64::k64_energy_query<<<1, 32, 0, ctx->stream>>>(ctx->d, ctx->energy_blocks);
    CU_LAUNCH();
    mpr_status s = fetch_state64(ctx);
    if (s != MPR_OK) return s;
    *h_e = ctx->h_state.e_query;
    return MPR_OK;
}

mpr_status mpr64_get_transform(mpr64_ctx* ctx, double* h_zmin, double* h_zmax)
{
    if (!ctx || !h_zmin || !h_zmax) return MPR_ERR_ARG;
    *h_zmin = ctx->h_state.zmin; *h_zmax = ctx->h_state.zmax;      // fixed since mpr64_create, which fetched them
    return MPR_OK;
}

mpr_status mpr64_get_stats(mpr64_ctx* ctx, mpr_stats* o)
{
    if (!ctx || !o) return MPR_ERR_ARG;
    ENTER64(ctx);
    mpr_status s = fetch_state64(ctx);
    if (s != MPR_OK) return s;
    const mpr64::State64& g = ctx->h_state;
    o->equil_sweeps = g.i; o->t = g.t; o->equilibrated = g.done; o->realizations = g.realizations;
    o->n_free = g.n_free; o->n_samples = g.n_samples; o->n_bonds = (uint64_t)ctx->d.n_bonds;
    o->a = g.a; o->k = g.k; o->A_last = g.A_last; o->e_last = g.e_last;
    o->z_min = (float)g.zmin; o->z_max = (float)g.zmax;
    return MPR_OK;
}

mpr_status mpr64_get_launch_count(mpr64_ctx* ctx, uint64_t* h_count)
{
    if (!ctx || !h_count) return MPR_ERR_ARG;
    *h_count = ctx->launches;
    return MPR_OK;
}

}  // extern "C"
