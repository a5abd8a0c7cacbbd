// mpr_microbench.cu -- measured denominators of the sweep kernel's roofline:
// the special-function (MUFU) rate north_star's "transcendental work at SFU peak" is divided by, and the issue and
// pipe rates DESIGN.md section 6 quotes.  Built into libmpr_microbench.so (not part of the MPR library); run by
// `python bench.py --sfu-peak`.  Every kernel is a register-only loop of independent dependency chains, long enough
// that launch overhead is below 1 %; the host times it with CUDA events and returns thread-level results per second.
#include <cstdint>
#include <cuda_runtime.h>

namespace {

constexpr int CHAINS = 8;      // independent chains per thread (latency hidden by ILP and by 64 warps / SM)

enum Op { OP_EX2 = 0, OP_RCP = 1, OP_FFMA = 2, OP_FFMA2 = 3, OP_IMAD_WIDE = 4, OP_LOP3 = 5, OP_IMAD = 6,
          OP_MUL_WIDE_ONLY = 7, OP_MUL_HI = 8, OP_PHILOX = 9, OP_LDS64 = 10 };

// Philox4x32-10 (Salmon et al., SC'11) as the sweep kernel computes it: 2 wide multiplies and 2 three-input XORs per round
__device__ __forceinline__ void philox_rounds(uint32_t& c0, uint32_t& c1, uint32_t& c2, uint32_t& c3, uint32_t k0, uint32_t k1)
{
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint64_t p0 = (uint64_t)c0 * 0xD2511F53u, p1 = (uint64_t)c2 * 0xCD9E8D57u;
        const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ (k0 + (uint32_t)r * 0x9E3779B9u);
        const uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ (k1 + (uint32_t)r * 0xBB67AE85u);
        c0 = n0; c1 = (uint32_t)p1; c2 = n2; c3 = (uint32_t)p0;
    }
}

template <int OP>
__global__ void __launch_bounds__(1024) k_chain(uint32_t iters, float seed, float* __restrict__ sink)
{
    float x[CHAINS];
    uint32_t u[CHAINS];
    uint64_t w[CHAINS];
    float2 p[CHAINS];
#pragma unroll
    for (int c = 0; c < CHAINS; ++c) {
        x[c] = seed + 1e-3f * (float)(threadIdx.x + c);
        u[c] = (uint32_t)threadIdx.x * 2654435761u + (uint32_t)c;
        w[c] = u[c];
        p[c] = make_float2(x[c], -x[c]);
    }
#pragma unroll 1
    for (uint32_t i = 0; i < iters; ++i) {
#pragma unroll
        for (int c = 0; c < CHAINS; ++c) {
            if (OP == OP_EX2) asm volatile("ex2.approx.ftz.f32 %0, %0;" : "+f"(x[c]));
            if (OP == OP_RCP) asm volatile("rcp.approx.ftz.f32 %0, %0;" : "+f"(x[c]));
            if (OP == OP_FFMA) asm volatile("fma.rn.f32 %0, %0, %1, %1;" : "+f"(x[c]) : "f"(seed));
            if (OP == OP_FFMA2) {
                uint64_t& q = reinterpret_cast<uint64_t&>(p[c]);
                const uint64_t s = reinterpret_cast<const uint64_t&>(p[(c + 1) % CHAINS]);
                asm volatile("fma.rn.f32x2 %0, %0, %1, %1;" : "+l"(q) : "l"(s));
            }
            if (OP == OP_IMAD_WIDE) asm volatile("mul.wide.u32 %0, %1, 0xD2511F53;\n\txor.b32 %1, %1, %2;" : "=l"(w[c]), "+r"(u[c]) : "r"((uint32_t)(w[c] >> 32)));
            if (OP == OP_LOP3) asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(u[c]) : "r"(i), "r"(u[(c + 1) % CHAINS]));
            if (OP == OP_IMAD) asm volatile("mad.lo.u32 %0, %0, %1, %2;" : "+r"(u[c]) : "r"(0x9E3779B9u), "r"(i));
            if (OP == OP_MUL_WIDE_ONLY) asm volatile("{\n\t.reg .b32 lo, hi;\n\tmov.b64 {lo, hi}, %0;\n\tmul.wide.u32 %0, hi, 0xD2511F53;\n\t}" : "+l"(w[c]));
            if (OP == OP_MUL_HI) asm volatile("mul.hi.u32 %0, %0, 0xD2511F53;" : "+r"(u[c]));
            if (OP == OP_PHILOX && c < 4) {        // four calls in flight per thread; a "result" = one call (4 words)
                uint32_t c1 = i, c2 = 2u, c3 = (uint32_t)c;
                philox_rounds(u[c], c1, c2, c3, 0x1234567u, 0x89ABCDEFu);
                u[c] ^= c1 ^ c2 ^ c3;
            }
            if (OP == OP_LDS64) {                   // a "result" = one conflict-free 64-bit shared-memory load per thread
                extern __shared__ float2 s_buf[];
                const float2 v = s_buf[(u[c] + (uint32_t)threadIdx.x) & 1023u];
                u[c] += __float_as_uint(v.x) + 1024u;
            }
        }
    }
    float acc = 0.0f;
#pragma unroll
    for (int c = 0; c < CHAINS; ++c) acc += x[c] + (float)u[c] + (float)(uint32_t)w[c] + p[c].x + p[c].y;
    if (acc == 12345.678f) sink[0] = acc;      // never true: keeps the chains alive
}

template <int OP>
double run(uint32_t iters, int blocks, cudaStream_t s, float* sink)
{
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    const size_t smem = OP == OP_LDS64 ? 1024 * sizeof(float2) : 0;
    if (OP == OP_PHILOX) iters /= 16;                                          // a call is 40 instructions
    k_chain<OP><<<blocks, 1024, smem, s>>>(iters / 8 + 1, 0.5f, sink);       // warm-up
    cudaEventRecord(e0, s);
    k_chain<OP><<<blocks, 1024, smem, s>>>(iters, 0.5f, sink);
    cudaEventRecord(e1, s);
    cudaEventSynchronize(e1);
    float ms = 0.0f;
    cudaEventElapsedTime(&ms, e0, e1);
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    if (cudaGetLastError() != cudaSuccess || ms <= 0.0f) return -1.0;
    // the IMAD.WIDE chain carries one XOR per multiply (Philox's round shape): count the multiplies only
    return (double)iters * (OP == OP_PHILOX ? 4 : CHAINS) * 1024.0 * (double)blocks / ((double)ms * 1e-3);
}

}  // namespace

extern "C" {

// Thread-level results per second of one operation issued back to back from every SM (blocks = 2 x SM count of
// 1024 threads).  op: 0 ex2.approx (MUFU), 1 rcp.approx (MUFU), 2 FFMA, 3 FFMA2 (counted as instructions, two fp32
// results each), 4 IMAD.WIDE (+ one LOP), 5 LOP3, 6 IMAD, 7 IMAD.WIDE alone, 8 IMAD.HI, 9 whole Philox4x32-10 calls,
// 10 conflict-free LDS.64.  h_per_s receives the rate; returns 0 on success.
int mprbench_rate(int op, uint32_t iters, double* h_per_s, int* h_sm_count)
{
    if (!h_per_s || !h_sm_count || iters == 0) return 1;
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return 2;
    float* sink = nullptr;
    if (cudaMalloc(&sink, 256) != cudaSuccess) return 2;
    const int blocks = 2 * sms;
    double r = -1.0;
    switch (op) {
    case OP_EX2: r = run<OP_EX2>(iters, blocks, 0, sink); break;
    case OP_RCP: r = run<OP_RCP>(iters, blocks, 0, sink); break;
    case OP_FFMA: r = run<OP_FFMA>(iters, blocks, 0, sink); break;
    case OP_FFMA2: r = run<OP_FFMA2>(iters, blocks, 0, sink); break;
    case OP_IMAD_WIDE: r = run<OP_IMAD_WIDE>(iters, blocks, 0, sink); break;
    case OP_LOP3: r = run<OP_LOP3>(iters, blocks, 0, sink); break;
    case OP_IMAD: r = run<OP_IMAD>(iters, blocks, 0, sink); break;
    case OP_MUL_WIDE_ONLY: r = run<OP_MUL_WIDE_ONLY>(iters, blocks, 0, sink); break;
    case OP_MUL_HI: r = run<OP_MUL_HI>(iters, blocks, 0, sink); break;
    case OP_PHILOX: r = run<OP_PHILOX>(iters, blocks, 0, sink); break;
    case OP_LDS64: r = run<OP_LDS64>(iters, blocks, 0, sink); break;
    default: cudaFree(sink); return 1;
    }
    cudaFree(sink);
    if (r < 0.0) return 2;
    *h_per_s = r; *h_sm_count = sms;
    return 0;
}

}  // extern "C"
