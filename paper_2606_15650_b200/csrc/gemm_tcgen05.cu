// gemm_tcgen05.cu -- K2: C[M,N] = A[M,K] * W[N,K]^T (+bias, +GELU | +residual) for the encoder's dense
// projections (S8a A2, A4, A5, A6; BJ "tcgen05/TMEM tensor-core GEMMs fed by TMA").
//
// sm_100a design: persistent CTAs (one per SM), warp-specialised:
//   warp 0   TMA producer : cp.async.bulk.tensor 2-D tiles (128B swizzle) of A [128 x 64] and W [BN x 64]
//                           into a STAGES-deep shared-memory ring, completion on mbarriers
//   warp 1   MMA issuer   : one thread issues tcgen05.mma (M=128, N=BN, K=16, BF16 -> FP32) with shared-memory
//                           matrix descriptors; accumulators live in TMEM, double-buffered (2 x BN columns) so
//                           the epilogue of tile i overlaps the mainloop of tile i+1; tcgen05.commit frees
//                           ring slots / publishes accumulators
//   warp 2   TMEM allocator
//   warps 4-7 epilogue    : tcgen05.ld (32 lanes x 32 columns per warp) -> bias / GELU / residual in
//                           registers -> vectorised global stores
// Operands are "TN": A row-major [M,K], W row-major [N,K] (both K-contiguous = K-major UMMA operands).
#include "common.cuh"
#include "ptx_sm100.cuh"

#include <cuda.h>

namespace {

constexpr int BM = 128;
constexpr int BK = 64;                    // 64 BF16 = 128 bytes = one swizzle row
constexpr int UMMA_K = 16;
constexpr int kThreads = 256;
constexpr int A_STAGE_BYTES = BM * BK * 2;

template <int BN> struct Cfg {
    static constexpr int B_STAGE_BYTES = BN * BK * 2;
    static constexpr int STAGE_BYTES = A_STAGE_BYTES + B_STAGE_BYTES;
    static constexpr int STAGES = (BN == 256) ? 4 : 6;
    static constexpr int TMEM_COLS = 2 * BN;      // two accumulator buffers
    static constexpr int SMEM_BYTES = STAGES * STAGE_BYTES + 1024 /*align slack*/ + 256 /*barriers*/;
};

// erf-GELU with the Abramowitz-Stegun 7.1.26 rational-exponential form (|err(erf)| < 1.5e-7, far below
// the BF16 rounding of the stored activation); 2 MUFU ops + ~12 FMA-pipe ops per element.
__device__ __forceinline__ float gelu_fast(float z) {
    const float x = fabsf(z) * 0.70710678118654752f;
    const float t = __fdividef(1.0f, fmaf(0.3275911f, x, 1.0f));
    float p = fmaf(t, 1.061405429f, -1.453152027f);
    p = fmaf(t, p, 1.421413741f);
    p = fmaf(t, p, -0.284496736f);
    p = fmaf(t, p, 0.254829592f);
    p *= t;
    const float e = __expf(-x * x);
    const float erf_abs = fmaf(-p, e, 1.0f);
    return 0.5f * z * (1.0f + copysignf(erf_abs, z));
}

__device__ __forceinline__ uint32_t pack_bf16(float a, float b) {
    __nv_bfloat162 v = __floats2bfloat162_rn(a, b);
    return *reinterpret_cast<uint32_t*>(&v);
}

// EPI: 0 = +bias -> BF16;  1 = +bias, GELU -> BF16;  2 = +bias +residual(FP32) -> FP32
template <int BN, int EPI>
__global__ void __launch_bounds__(kThreads, 1)
gemm_bf16_tcgen05_kernel(const __grid_constant__ CUtensorMap tmap_a, const __grid_constant__ CUtensorMap tmap_b,
                         const float* __restrict__ bias, const float* __restrict__ residual, void* __restrict__ Cout,
                         int M, int N, int K)
{
    using C = Cfg<BN>;
    extern __shared__ uint8_t smem_raw[];
    const uint32_t smem_base = (ptx::smem_u32(smem_raw) + 1023u) & ~1023u;
    const uint32_t bar_base = smem_base + C::STAGES * C::STAGE_BYTES;
    auto full_bar = [&](int s) { return bar_base + 8u * s; };
    auto empty_bar = [&](int s) { return bar_base + 8u * (C::STAGES + s); };
    auto tfull_bar = [&](int a) { return bar_base + 8u * (2 * C::STAGES + a); };
    auto tempty_bar = [&](int a) { return bar_base + 8u * (2 * C::STAGES + 2 + a); };
    const uint32_t tmem_slot = bar_base + 8u * (2 * C::STAGES + 4);
    uint32_t* tmem_slot_ptr = reinterpret_cast<uint32_t*>(smem_raw + (tmem_slot - ptx::smem_u32(smem_raw)));

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int num_m = (M + BM - 1) / BM, num_n = (N + BN - 1) / BN;
    const int num_tiles = num_m * num_n;
    const int num_kb = K / BK;

    if (warp == 0 && lane == 0) {
        ptx::prefetch_tensormap(&tmap_a);
        ptx::prefetch_tensormap(&tmap_b);
    }
    if (warp == 1 && lane == 0) {
        for (int s = 0; s < C::STAGES; s++) { ptx::mbar_init(full_bar(s), 1); ptx::mbar_init(empty_bar(s), 1); }
        for (int a = 0; a < 2; a++) { ptx::mbar_init(tfull_bar(a), 1); ptx::mbar_init(tempty_bar(a), 4); }
        ptx::fence_barrier_init();
        ptx::fence_proxy_async();
    }
    if (warp == 2) {
        ptx::tmem_alloc(tmem_slot, C::TMEM_COLS);
        ptx::tmem_relinquish();
    }
    ptx::tc_fence_before();
    __syncthreads();
    ptx::tc_fence_after();
    const uint32_t tmem_base = *tmem_slot_ptr;

    if (warp == 0) {
        if (lane == 0) {
            int s = 0; uint32_t ph = 0;
            for (int tile = blockIdx.x; tile < num_tiles; tile += gridDim.x) {
                const int m_blk = tile / num_n, n_blk = tile % num_n;
                for (int kb = 0; kb < num_kb; kb++) {
                    ptx::mbar_wait(empty_bar(s), ph ^ 1u);
                    ptx::mbar_arrive_expect_tx(full_bar(s), C::STAGE_BYTES);
                    const uint32_t sa = smem_base + s * C::STAGE_BYTES;
                    ptx::tma_load_2d(sa, &tmap_a, full_bar(s), kb * BK, m_blk * BM);
                    ptx::tma_load_2d(sa + A_STAGE_BYTES, &tmap_b, full_bar(s), kb * BK, n_blk * BN);
                    if (++s == C::STAGES) { s = 0; ph ^= 1u; }
                }
            }
        }
    } else if (warp == 1) {
        if (lane == 0) {
            constexpr uint32_t idesc = ptx::make_idesc_bf16(BM, BN);
            int s = 0; uint32_t ph = 0;
            int acc = 0; uint32_t acc_ph = 0;
            for (int tile = blockIdx.x; tile < num_tiles; tile += gridDim.x) {
                ptx::mbar_wait(tempty_bar(acc), acc_ph ^ 1u);
                ptx::tc_fence_after();
                const uint32_t d_tmem = tmem_base + (uint32_t)(acc * BN);
                for (int kb = 0; kb < num_kb; kb++) {
                    ptx::mbar_wait(full_bar(s), ph);
                    ptx::tc_fence_after();
                    const uint32_t sa = smem_base + s * C::STAGE_BYTES;
                    const uint64_t adesc = ptx::make_desc_k_sw128(sa);
                    const uint64_t bdesc = ptx::make_desc_k_sw128(sa + A_STAGE_BYTES);
#pragma unroll
                    for (int k = 0; k < BK / UMMA_K; k++) {
                        // +32 bytes along K inside the 128-byte swizzle row = +2 in the (addr >> 4) field
                        ptx::mma_f16_ss(d_tmem, adesc + (uint64_t)(2 * k), bdesc + (uint64_t)(2 * k), idesc,
                                        (kb | k) ? 1u : 0u);
                    }
                    ptx::mma_commit(empty_bar(s));
                    if (++s == C::STAGES) { s = 0; ph ^= 1u; }
                }
                ptx::mma_commit(tfull_bar(acc));
                if (++acc == 2) { acc = 0; acc_ph ^= 1u; }
            }
        }
    } else if (warp >= 4) {
        const int q = warp & 3;                       // TMEM lane quarter this warp may access
        int acc = 0; uint32_t acc_ph = 0;
        for (int tile = blockIdx.x; tile < num_tiles; tile += gridDim.x) {
            const int m_blk = tile / num_n, n_blk = tile % num_n;
            const int row = m_blk * BM + q * 32 + lane;
            ptx::mbar_wait(tfull_bar(acc), acc_ph);
            ptx::tc_fence_after();
            const uint32_t t_base = tmem_base + ((uint32_t)(q * 32) << 16) + (uint32_t)(acc * BN);
#pragma unroll 1
            for (int c0 = 0; c0 < BN; c0 += 32) {
                uint32_t r[32];
                ptx::tmem_ld_32x32b_x32(t_base + (uint32_t)c0, r);
                ptx::tmem_ld_wait();
                const int col = n_blk * BN + c0;
                if (row < M && col < N) {
                    if (col + 32 <= N) {
                        const float4* b4 = reinterpret_cast<const float4*>(bias + col);
                        if (EPI == 2) {
                            const float4* r4 = reinterpret_cast<const float4*>(residual + (size_t)row * N + col);
                            float4* o4 = reinterpret_cast<float4*>(reinterpret_cast<float*>(Cout) + (size_t)row * N + col);
#pragma unroll
                            for (int v = 0; v < 8; v++) {
                                const float4 b = __ldg(b4 + v), x = __ldg(r4 + v);
                                float4 o;
                                o.x = __uint_as_float(r[4 * v + 0]) + b.x + x.x;
                                o.y = __uint_as_float(r[4 * v + 1]) + b.y + x.y;
                                o.z = __uint_as_float(r[4 * v + 2]) + b.z + x.z;
                                o.w = __uint_as_float(r[4 * v + 3]) + b.w + x.w;
                                o4[v] = o;
                            }
                        } else {
                            uint4* o4 = reinterpret_cast<uint4*>(reinterpret_cast<__nv_bfloat16*>(Cout) + (size_t)row * N + col);
#pragma unroll
                            for (int v = 0; v < 4; v++) {
                                const float4 b0 = __ldg(b4 + 2 * v), b1 = __ldg(b4 + 2 * v + 1);
                                float f[8];
                                f[0] = __uint_as_float(r[8 * v + 0]) + b0.x; f[1] = __uint_as_float(r[8 * v + 1]) + b0.y;
                                f[2] = __uint_as_float(r[8 * v + 2]) + b0.z; f[3] = __uint_as_float(r[8 * v + 3]) + b0.w;
                                f[4] = __uint_as_float(r[8 * v + 4]) + b1.x; f[5] = __uint_as_float(r[8 * v + 5]) + b1.y;
                                f[6] = __uint_as_float(r[8 * v + 6]) + b1.z; f[7] = __uint_as_float(r[8 * v + 7]) + b1.w;
                                if (EPI == 1) {
#pragma unroll
                                    for (int u = 0; u < 8; u++) f[u] = gelu_fast(f[u]);
                                }
                                o4[v] = make_uint4(pack_bf16(f[0], f[1]), pack_bf16(f[2], f[3]),
                                                   pack_bf16(f[4], f[5]), pack_bf16(f[6], f[7]));
                            }
                        }
                    } else {
                        for (int u = 0; u < 32 && col + u < N; u++) {          // ragged N tail
                            float f = __uint_as_float(r[u]) + bias[col + u];
                            if (EPI == 1) f = gelu_fast(f);
                            if (EPI == 2) {
                                f += residual[(size_t)row * N + col + u];
                                reinterpret_cast<float*>(Cout)[(size_t)row * N + col + u] = f;
                            } else {
                                reinterpret_cast<__nv_bfloat16*>(Cout)[(size_t)row * N + col + u] = __float2bfloat16_rn(f);
                            }
                        }
                    }
                }
            }
            ptx::tc_fence_before();
            __syncwarp();
            if (lane == 0) ptx::mbar_arrive(tempty_bar(acc));
            if (++acc == 2) { acc = 0; acc_ph ^= 1u; }
        }
    }

    ptx::tc_fence_before();
    __syncthreads();
    if (warp == 2) {
        ptx::tc_fence_after();
        ptx::tmem_dealloc(tmem_base, C::TMEM_COLS);
    }
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

int make_tmap_bf16_2d(anon_ctx* ctx, CUtensorMap* tm, const void* base, uint64_t rows, uint64_t cols, uint32_t box_rows) {
    if (!ctx->encode_tiled) {
        void* fn = nullptr;
        cudaDriverEntryPointQueryResult q;
        cudaError_t e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &q);
        if (e != cudaSuccess || q != cudaDriverEntryPointSuccess || !fn)
            return cuda_fail(ctx, e == cudaSuccess ? cudaErrorUnknown : e, "cudaGetDriverEntryPoint(cuTensorMapEncodeTiled)");
        ctx->encode_tiled = fn;
    }
    const cuuint64_t gdim[2] = {cols, rows};
    const cuuint64_t gstride[1] = {cols * 2};
    const cuuint32_t box[2] = {(cuuint32_t)BK, box_rows};
    const cuuint32_t estr[2] = {1, 1};
    CUresult r = ((EncodeTiledFn)ctx->encode_tiled)(tm, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<void*>(base), gdim,
                                                    gstride, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                                                    CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                                                    CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) {
        snprintf(ctx->cuda_err, sizeof ctx->cuda_err, "cuTensorMapEncodeTiled failed: CUresult %d", (int)r);
        return ANON_ERR_CUDA;
    }
    return ANON_OK;
}

template <int BN, int EPI>
int launch_gemm(anon_ctx* ctx, const __nv_bfloat16* A, const __nv_bfloat16* W, const float* bias, const float* residual,
                void* Cout, int M, int N, int K)
{
    using C = Cfg<BN>;
    CUtensorMap ta, tb;
    int rc = make_tmap_bf16_2d(ctx, &ta, A, (uint64_t)M, (uint64_t)K, BM);
    if (rc) return rc;
    rc = make_tmap_bf16_2d(ctx, &tb, W, (uint64_t)N, (uint64_t)K, BN);
    if (rc) return rc;
    auto kern = gemm_bf16_tcgen05_kernel<BN, EPI>;
    static bool attr_set = false;
    if (!attr_set) {
        CU_TRY(ctx, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, C::SMEM_BYTES));
        attr_set = true;
    }
    const int tiles = ((M + BM - 1) / BM) * ((N + BN - 1) / BN);
    const int grid = tiles < ctx->sm_count ? tiles : ctx->sm_count;
    kern<<<grid, kThreads, C::SMEM_BYTES, ctx->stream>>>(ta, tb, bias, residual, Cout, M, N, K);
    CU_LAUNCH_CHECK(ctx, "gemm_bf16_tcgen05_kernel");
    return ANON_OK;
}

}  // namespace

int gemm_bf16_impl(anon_ctx* ctx, const __nv_bfloat16* A, const __nv_bfloat16* W, const float* bias,
                   const float* residual, void* Cout, int M, int N, int K, int epilogue)
{
    if (!ctx || !A || !W || !bias || !Cout || M < 0 || N <= 0 || K <= 0 || epilogue < 0 || epilogue > 2 ||
        (epilogue == 2 && !residual))
        return ANON_ERR_INVALID_ARG;
    if (K % BK != 0 || N % 8 != 0) return ANON_ERR_UNSUPPORTED;
    if (M == 0) return ANON_OK;
    if (N > 128) {
        switch (epilogue) {
            case 0: return launch_gemm<256, 0>(ctx, A, W, bias, residual, Cout, M, N, K);
            case 1: return launch_gemm<256, 1>(ctx, A, W, bias, residual, Cout, M, N, K);
            default: return launch_gemm<256, 2>(ctx, A, W, bias, residual, Cout, M, N, K);
        }
    }
    switch (epilogue) {
        case 0: return launch_gemm<128, 0>(ctx, A, W, bias, residual, Cout, M, N, K);
        case 1: return launch_gemm<128, 1>(ctx, A, W, bias, residual, Cout, M, N, K);
        default: return launch_gemm<128, 2>(ctx, A, W, bias, residual, Cout, M, N, K);
    }
}

extern "C" int anon_gemm_bf16(anon_ctx* ctx, const void* d_A, const void* d_W, const float* d_bias,
                              const float* d_residual, void* d_C, int32_t M, int32_t N, int32_t K, int32_t epilogue)
{
    if (!ctx) return ANON_ERR_INVALID_ARG;
    CU_TRY(ctx, cudaSetDevice(ctx->device));
    return gemm_bf16_impl(ctx, (const __nv_bfloat16*)d_A, (const __nv_bfloat16*)d_W, d_bias, d_residual, d_C, M, N, K,
                          epilogue);
}
