// mpr_noalloc.inl -- ONE entry point that allocates nothing (include/mpr.h, "allocation-free entry point"), for callers that
// cannot call cudaMalloc and cannot hand over a workspace either: code under CUDA graph capture, tight serving loops,
// harnesses that forbid allocation.  Included at the end of mpr_api.cu (same translation unit: the static array below, the
// kernel that names it, the set-up that asks for its address and the entry point all live in this one .cu file).
//
// What it computes: the energy per bond e = H / N_GP of Eq. 2 of an angle field the caller holds in
// device memory -- the quantity Alg. 2 step 5.3 tracks (L199) -- i.e. mpr_energy without a context.  The existing path
// (k_energy + k_energy_query) keeps its per-block partial sums in the caller's workspace; this variant keeps one partial
// per grid row in a file-scope array of a fixed, modest size.

namespace {

constexpr int NOALLOC_MAX_ROWS = MPR_NOALLOC_MAX_ROWS;     // one double per row: 128 KB
constexpr int NOALLOC_THREADS  = 256;
constexpr int NOALLOC_BLOCKS   = 592;                      // 4 x 148 SMs, rows dealt over them

// The scratch: every GPU that loads the library holds these 128 KB + 256 B until exit.  Every call shares it, and it
// keeps the last call's contents: the row partials are all overwritten before they are read (rows of this call only),
// the ticket counter must start at zero and is cleared by the entry point before every launch (and left at zero by the
// kernel).  Calls that overlap on the GPU (two streams, two threads) race on it.
struct __align__(256) NoallocScratch {
    double       row_partial[NOALLOC_MAX_ROWS];
    unsigned int ticket;                                   // blocks of the running call that have delivered their rows
};
static __device__ __align__(256) NoallocScratch g_noalloc_scratch;

// H = - sum over the bonds of cos q(phi_i - phi_j), open boundaries: row r takes its right and its down bonds.  One
// partial per row in double (fixed order within a row: strided per thread, shuffle tree per warp, warps in order); the
// block that delivers last sums the rows' partials in the same fixed way and writes e = H / N_GP.  Bitwise reproducible.
__global__ void __launch_bounds__(NOALLOC_THREADS) k_energy_of_angles_noalloc(NoallocScratch* __restrict__ scratch,
                                                                              const float* __restrict__ phi, int rows, int cols,
                                                                              double q, double* __restrict__ d_e_per_bond)
{
    __shared__ double warp_part[NOALLOC_THREADS / 32];
    __shared__ unsigned int s_last;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    auto block_sum = [&](double x) {           // every thread calls it; thread 0 gets the sum
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) x += __shfl_xor_sync(0xFFFFFFFFu, x, o);
        __syncthreads();                       // warp_part is free again
        if (lane == 0) warp_part[warp] = x;
        __syncthreads();
        double t = 0.0;
        if (threadIdx.x == 0)
            for (int w = 0; w < NOALLOC_THREADS / 32; ++w) t += warp_part[w];
        return t;
    };
    for (int r = blockIdx.x; r < rows; r += gridDim.x) {
        const float* row = phi + (size_t)r * cols;
        double part = 0.0;
        for (int c = threadIdx.x; c < cols; c += NOALLOC_THREADS) {
            const double p = (double)row[c];
            if (c + 1 < cols) part -= cos(q * (p - (double)row[c + 1]));
            if (r + 1 < rows) part -= cos(q * (p - (double)row[c + cols]));
        }
        const double t = block_sum(part);
        if (threadIdx.x == 0) scratch->row_partial[r] = t;
    }
    if (threadIdx.x == 0) {
        __threadfence();                       // this block's partials before its ticket
        s_last = atomicAdd(&scratch->ticket, 1u) == gridDim.x - 1u ? 1u : 0u;
    }
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    double part = 0.0;
    for (int r = threadIdx.x; r < rows; r += NOALLOC_THREADS) part += __ldcg(&scratch->row_partial[r]);
    const double H = block_sum(part);
    if (threadIdx.x == 0) {
        const double n_bonds = (double)rows * (cols - 1) + (double)cols * (rows - 1);
        d_e_per_bond[0] = H / n_bonds;
        scratch->ticket = 0u;                  // as the next call wants it (the entry point clears it too)
    }
}

// Set-up, once per device, with that device current: in host code `g_noalloc_scratch` is a host-side stand-in for the
// array, not its device address -- the address comes from cudaGetSymbolAddress.
std::mutex g_noalloc_lock;
NoallocScratch* g_noalloc_ptr[64] = {};

mpr_status noalloc_scratch_of(int device, NoallocScratch** out)
{
    if (device < 0 || device >= 64) return MPR_ERR_ARG;
    std::lock_guard<std::mutex> hold(g_noalloc_lock);
    if (!g_noalloc_ptr[device]) {
        NoallocScratch* p = nullptr;
        if (!cuda_ok(cudaGetSymbolAddress((void**)&p, g_noalloc_scratch), "cudaGetSymbolAddress(g_noalloc_scratch)") || !p) return MPR_ERR_CUDA;
        g_noalloc_ptr[device] = p;
    }
    *out = g_noalloc_ptr[device];
    return MPR_OK;
}

}  // namespace

extern "C" {

mpr_status mpr_energy_of_angles_noalloc(const float* d_phi, int rows, int cols, double q, double* d_e_per_bond, void* cuda_stream)
{
    if (!d_phi || !d_e_per_bond || rows < 2 || cols < 2 || cols > 65534 || !(q > 0.0 && q <= 0.5)) return MPR_ERR_ARG;
    if (rows > NOALLOC_MAX_ROWS) {
        snprintf(g_cuda_err, sizeof g_cuda_err, "mpr_energy_of_angles_noalloc: %d rows exceed MPR_NOALLOC_MAX_ROWS = %d (the static scratch holds one partial per row)",
                 rows, NOALLOC_MAX_ROWS);
        return MPR_ERR_TOO_LARGE;
    }
    cudaPointerAttributes attr;
    if (!cuda_ok(cudaPointerGetAttributes(&attr, d_phi), "cudaPointerGetAttributes") || attr.type != cudaMemoryTypeDevice) return MPR_ERR_ARG;
    CU(cudaSetDevice(attr.device));
    NoallocScratch* scratch = nullptr;
    mpr_status s = noalloc_scratch_of(attr.device, &scratch);
    if (s != MPR_OK) return s;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    CU(cudaMemsetAsync(&scratch->ticket, 0, sizeof(unsigned int), st));       // must start at zero whatever the last call left
    const int blocks = rows < NOALLOC_BLOCKS ? rows : NOALLOC_BLOCKS;
    k_energy_of_angles_noalloc<<<blocks, NOALLOC_THREADS, 0, st>>>(scratch, d_phi, rows, cols, q, d_e_per_bond);
    CU(cudaGetLastError());
    return MPR_OK;
}

}  // extern "C"
