// microbench.cu -- measured issue-rate peaks for the two non-tensor, non-HBM bounds the hot path runs against
// (SURVEY.md §8(d) ¶1 and Appendix C: "Integer-ALU and MUFU rates are not in MEASURED_PEAKS.json -- measure"):
//   * the integer ALU pipe (LOP3 / SHF / IADD3), the bound of HMAC-SHA256 (K10);
//   * the MUFU pipe (ex2.approx), the co-limiter of attention at d_head = 64 (K3).
// Dependency-free in the sense of the survey: every thread runs 8 INDEPENDENT chains (the ALU pipe's latency is ~4-5
// issue slots), the SMs are fully occupied (2,048 threads each), no memory traffic inside the timed loop.  The result
// of every chain is folded into one store at the end so that nothing is optimised away.
#include "common.cuh"

namespace {

constexpr int kChains = 8;
constexpr int kUnroll = 16;

__device__ __forceinline__ uint32_t lop3_xor_and_or(uint32_t a, uint32_t b, uint32_t c) {
    uint32_t d; asm volatile("lop3.b32 %0, %1, %2, %3, 0x96;" : "=r"(d) : "r"(a), "r"(b), "r"(c)); return d;     // a ^ b ^ c
}
__device__ __forceinline__ uint32_t shf_l(uint32_t lo, uint32_t hi, uint32_t n) {
    uint32_t d; asm volatile("shf.l.wrap.b32 %0, %1, %2, %3;" : "=r"(d) : "r"(lo), "r"(hi), "r"(n)); return d;
}
__device__ __forceinline__ uint32_t iadd3(uint32_t a, uint32_t b, uint32_t c) {
    uint32_t d; asm volatile("{.reg .u32 t; add.u32 t, %1, %2; add.u32 %0, t, %3;}" : "=r"(d) : "r"(a), "r"(b), "r"(c)); return d;
}
__device__ __forceinline__ float ex2(float x) { float y; asm volatile("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }

// MODE 0: LOP3 + SHF + IADD3 per chain step (the SHA-256 mix); 1: LOP3 only; 2: SHF only; 3: IADD3 only; 4: ex2.approx
template <int MODE>
__global__ void __launch_bounds__(256) issue_rate_kernel(int iters, uint32_t seed, uint32_t* out)
{
    uint32_t v[kChains];
    float f[kChains];
#pragma unroll
    for (int c = 0; c < kChains; c++) { v[c] = seed * (threadIdx.x + 1u) + 0x9E3779B9u * c; f[c] = -1.0f - 0.001f * (float)(c + (threadIdx.x & 7)); }
    const uint32_t k1 = seed | 1u, k2 = seed ^ 0x5bd1e995u;
    for (int it = 0; it < iters; it++) {
#pragma unroll
        for (int u = 0; u < kUnroll; u++) {
#pragma unroll
            for (int c = 0; c < kChains; c++) {
                // the second operand is the neighbouring chain's value: a true three-register LOP3 / funnel SHF / IADD3 that
                // ptxas cannot fold into a cheaper form (a rotate of one register becomes LEA.HI, an add of two loop
                // constants becomes one IMAD.IADD on the FMA pipe); the 8 updates of one step stay independent of each other
                const uint32_t nb = v[(c + 1) & (kChains - 1)];
                if (MODE == 0) { v[c] = lop3_xor_and_or(v[c], nb, k2); v[c] = shf_l(v[c], nb, 7); v[c] = iadd3(v[c], nb, k1); }
                if (MODE == 1) v[c] = lop3_xor_and_or(v[c], nb, k2);
                if (MODE == 2) v[c] = shf_l(v[c], nb, 7);
                if (MODE == 3) v[c] = iadd3(v[c], nb, k1);
                if (MODE == 4) f[c] = ex2(f[c]);          // stays in (0, 1]: 2^x of a value in [-2, 1] ... converges, never denormal
            }
        }
    }
    uint32_t acc = 0;
#pragma unroll
    for (int c = 0; c < kChains; c++) acc ^= v[c] ^ __float_as_uint(f[c]);
    if (acc == 0x12345678u) out[blockIdx.x] = acc;          // practically never true: keeps the chains alive
}

template <int MODE>
int run_mode(anon_ctx* ctx, int iters, double ops_per_step, double* ops_per_s, double* ms_out)
{
    uint32_t* d_out = (uint32_t*)(ctx->d_status + 32);      // scratch words inside the 256-byte status allocation
    const int grid = ctx->sm_count * 8;                     // 8 CTAs x 256 threads = 2,048 threads per SM
    cudaEvent_t a, b;
    CU_TRY(ctx, cudaEventCreate(&a));
    CU_TRY(ctx, cudaEventCreate(&b));
    issue_rate_kernel<MODE><<<grid, 256, 0, ctx->stream>>>(iters / 8 + 1, 12345u, d_out);      // warm-up
    float best = 1e30f;
    for (int rep = 0; rep < 3; rep++) {
        cudaEventRecord(a, ctx->stream);
        issue_rate_kernel<MODE><<<grid, 256, 0, ctx->stream>>>(iters, 12345u + rep, d_out);
        cudaEventRecord(b, ctx->stream);
        cudaError_t e = cudaEventSynchronize(b);
        if (e != cudaSuccess) { cudaEventDestroy(a); cudaEventDestroy(b); return cuda_fail(ctx, e, "issue_rate_kernel"); }
        float ms = 0.f;
        cudaEventElapsedTime(&ms, a, b);
        if (ms < best) best = ms;
    }
    cudaEventDestroy(a); cudaEventDestroy(b);
    const double threads = (double)grid * 256.0;
    *ops_per_s = threads * (double)iters * kUnroll * kChains * ops_per_step / (best * 1e-3);
    if (ms_out) *ms_out = best;
    return ANON_OK;
}

}  // namespace

extern "C" int anon_microbench(anon_ctx* ctx, int32_t mode, int32_t iters, double* thread_ops_per_s, double* kernel_ms)
{
    if (!ctx || !thread_ops_per_s || iters <= 0 || iters > (1 << 20)) return ANON_ERR_INVALID_ARG;
    CU_TRY(ctx, cudaSetDevice(ctx->device));
    switch (mode) {
        case 0: return run_mode<0>(ctx, iters, 3.0, thread_ops_per_s, kernel_ms);
        case 1: return run_mode<1>(ctx, iters, 1.0, thread_ops_per_s, kernel_ms);
        case 2: return run_mode<2>(ctx, iters, 1.0, thread_ops_per_s, kernel_ms);
        case 3: return run_mode<3>(ctx, iters, 1.0, thread_ops_per_s, kernel_ms);     // one IADD3 in the SASS
        case 4: return run_mode<4>(ctx, iters, 1.0, thread_ops_per_s, kernel_ms);
        default: return ANON_ERR_INVALID_ARG;
    }
}
