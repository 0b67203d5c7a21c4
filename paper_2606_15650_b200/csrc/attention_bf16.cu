// attention_bf16.cu -- K3: packed variable-length bidirectional self-attention, d_head = 64 (S8a A3; S8c O1).
// No padding FLOPs: the work list holds one item per (sequence, 64-query tile), longest sequences first;
// keys are walked in 64-key tiles up to the sequence's own length only.  BF16 operands, FP32 scores,
// FP32 online softmax (exp2 with the 1/sqrt(64)*log2(e) scale folded in), FP32 output accumulators.
//
// v0 (this file): warp-level mma.sync.m16n8k16 tensor-core tiles fed by cp.async double buffering and
// ldmatrix from XOR-swizzled shared memory.  The tcgen05/TMEM version replaces it once the GEMM path is tuned.
#include "common.cuh"

#include <algorithm>
#include <vector>

namespace {

constexpr int kQT = 64;     // queries per CTA (16 per warp)
constexpr int kKT = 64;     // keys per pipeline stage
constexpr int kD = 64;

struct WorkItem { int q_row0; int kv_row0; int n; int q_valid; };   // rows relative to the chunk

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void cp_async16(uint32_t dst, const void* src, int src_bytes) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(dst), "l"(src), "r"(src_bytes) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N> __device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }
__device__ __forceinline__ void ldsm_x4(uint32_t addr, uint32_t& r0, uint32_t& r1, uint32_t& r2, uint32_t& r3) {
    asm volatile("ldmatrix.sync.aligned.m8n8.x4.shared.b16 {%0,%1,%2,%3}, [%4];" : "=r"(r0), "=r"(r1), "=r"(r2), "=r"(r3) : "r"(addr));
}
__device__ __forceinline__ void ldsm_x4_t(uint32_t addr, uint32_t& r0, uint32_t& r1, uint32_t& r2, uint32_t& r3) {
    asm volatile("ldmatrix.sync.aligned.m8n8.x4.trans.shared.b16 {%0,%1,%2,%3}, [%4];" : "=r"(r0), "=r"(r1), "=r"(r2), "=r"(r3) : "r"(addr));
}
__device__ __forceinline__ void mma_bf16(float (&c)[4], const uint32_t (&a)[4], uint32_t b0, uint32_t b1) {
    asm volatile("mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
                 : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3])
                 : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1));
}
__device__ __forceinline__ uint32_t pack2(float a, float b) {
    __nv_bfloat162 v = __floats2bfloat162_rn(a, b);
    return *reinterpret_cast<uint32_t*>(&v);
}
// tile of 64 rows x 64 BF16 (128 B per row), 16-byte chunk index XOR-swizzled by (row & 7)
__device__ __forceinline__ uint32_t tile_off(int row, int chunk) { return (uint32_t)(row * 128 + ((chunk ^ (row & 7)) << 4)); }

// loads rows [row0, row0+64) x 64 columns starting at column col0 of a [*, ld] BF16 matrix; rows >= rows_valid zero-filled
__device__ __forceinline__ void load_tile(uint32_t smem, const __nv_bfloat16* base, size_t ld, int row0, int rows_valid, int col0, int tid) {
#pragma unroll
    for (int it = 0; it < 4; it++) {
        const int idx = tid + it * 128;          // 512 chunks of 16 B
        const int r = idx >> 3, c = idx & 7;
        const bool ok = r < rows_valid;
        const __nv_bfloat16* src = base + (size_t)(row0 + (ok ? r : 0)) * ld + col0 + c * 8;
        cp_async16(smem + tile_off(r, c), src, ok ? 16 : 0);
    }
}

__global__ void __launch_bounds__(128) attention_bf16_kernel(const __nv_bfloat16* __restrict__ qkv, const WorkItem* __restrict__ work,
                                                             int H, __nv_bfloat16* __restrict__ ctx)
{
    __shared__ __align__(128) uint8_t sQ[kQT * 128];
    __shared__ __align__(128) uint8_t sK[2][kKT * 128];
    __shared__ __align__(128) uint8_t sV[2][kKT * 128];
    const WorkItem w = work[blockIdx.x];
    const int head = blockIdx.y;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31, g = lane >> 2, t = lane & 3;
    const size_t ld = (size_t)3 * H;
    const int n = w.n;
    const int nkt = (n + kKT - 1) / kKT;

    load_tile(smem_u32(sQ), qkv, ld, w.q_row0, w.q_valid, head * kD, tid);
    load_tile(smem_u32(sK[0]), qkv, ld, w.kv_row0, n, H + head * kD, tid);
    load_tile(smem_u32(sV[0]), qkv, ld, w.kv_row0, n, 2 * H + head * kD, tid);
    cp_async_commit();

    uint32_t qf[4][4];
    float o[8][4];
#pragma unroll
    for (int i = 0; i < 8; i++) { o[i][0] = o[i][1] = o[i][2] = o[i][3] = 0.f; }
    float m_run[2] = {-INFINITY, -INFINITY}, l_run[2] = {0.f, 0.f};
    const float sl2 = 0.125f * 1.4426950408889634f;

    for (int kt = 0; kt < nkt; kt++) {
        const int buf = kt & 1;
        if (kt + 1 < nkt) {
            const int k0 = (kt + 1) * kKT;
            load_tile(smem_u32(sK[buf ^ 1]), qkv, ld, w.kv_row0 + k0, n - k0, H + head * kD, tid);
            load_tile(smem_u32(sV[buf ^ 1]), qkv, ld, w.kv_row0 + k0, n - k0, 2 * H + head * kD, tid);
            cp_async_commit();
            cp_async_wait<1>();
        } else {
            cp_async_wait<0>();
        }
        __syncthreads();
        if (kt == 0) {
#pragma unroll
            for (int kk = 0; kk < 4; kk++)
                ldsm_x4(smem_u32(sQ) + tile_off(warp * 16 + (lane & 15), 2 * kk + (lane >> 4)), qf[kk][0], qf[kk][1], qf[kk][2], qf[kk][3]);
        }
        // S = Q K^T : 16 x 64 per warp
        float s[8][4];
#pragma unroll
        for (int i = 0; i < 8; i++) { s[i][0] = s[i][1] = s[i][2] = s[i][3] = 0.f; }
        const uint32_t kb = smem_u32(sK[buf]);
#pragma unroll
        for (int kk = 0; kk < 4; kk++) {
#pragma unroll
            for (int np = 0; np < 4; np++) {            // pairs of 8-key tiles
                uint32_t b0, b1, b2, b3;
                // matrices: [keys 16np..+7, d 16kk..+7], [same keys, d +8], [keys +8, d], [keys +8, d +8]
                const int row = np * 16 + (lane & 7) + ((lane >> 4) << 3);
                const int chunk = 2 * kk + ((lane >> 3) & 1);
                ldsm_x4(kb + tile_off(row, chunk), b0, b1, b2, b3);
                mma_bf16(s[2 * np], qf[kk], b0, b1);
                mma_bf16(s[2 * np + 1], qf[kk], b2, b3);
            }
        }
        // mask keys past the end of the sequence (last tile only)
        const int kbase = kt * kKT;
        if (kbase + kKT > n) {
#pragma unroll
            for (int i = 0; i < 8; i++) {
                const int c = kbase + i * 8 + 2 * t;
                if (c >= n) { s[i][0] = -INFINITY; s[i][2] = -INFINITY; }
                if (c + 1 >= n) { s[i][1] = -INFINITY; s[i][3] = -INFINITY; }
            }
        }
        // online softmax for rows g (h=0) and g+8 (h=1)
#pragma unroll
        for (int h = 0; h < 2; h++) {
            float mx = -INFINITY;
#pragma unroll
            for (int i = 0; i < 8; i++) mx = fmaxf(mx, fmaxf(s[i][2 * h], s[i][2 * h + 1]));
            mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, 1));
            mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, 2));
            const float m_new = fmaxf(m_run[h], mx);
            const float corr = exp2f((m_run[h] - m_new) * sl2);
            m_run[h] = m_new;
            float sum = 0.f;
#pragma unroll
            for (int i = 0; i < 8; i++) {
                const float p0 = exp2f((s[i][2 * h] - m_new) * sl2), p1 = exp2f((s[i][2 * h + 1] - m_new) * sl2);
                s[i][2 * h] = p0; s[i][2 * h + 1] = p1;
                sum += p0 + p1;
            }
            l_run[h] = l_run[h] * corr + sum;
#pragma unroll
            for (int i = 0; i < 8; i++) { o[i][2 * h] *= corr; o[i][2 * h + 1] *= corr; }
        }
        // O += P V
        const uint32_t vb = smem_u32(sV[buf]);
#pragma unroll
        for (int kk = 0; kk < 4; kk++) {               // 16 keys per step
            uint32_t pa[4];
            pa[0] = pack2(s[2 * kk][0], s[2 * kk][1]);
            pa[1] = pack2(s[2 * kk][2], s[2 * kk][3]);
            pa[2] = pack2(s[2 * kk + 1][0], s[2 * kk + 1][1]);
            pa[3] = pack2(s[2 * kk + 1][2], s[2 * kk + 1][3]);
#pragma unroll
            for (int dp = 0; dp < 4; dp++) {           // pairs of 8-wide d tiles
                uint32_t b0, b1, b2, b3;
                // transposed loads: matrices [keys 16kk..+7, d 16dp..+7], [keys +8, d], [keys, d +8], [keys +8, d +8]
                const int row = kk * 16 + (lane & 7) + (((lane >> 3) & 1) << 3);
                const int chunk = 2 * dp + (lane >> 4);
                ldsm_x4_t(vb + tile_off(row, chunk), b0, b1, b2, b3);
                mma_bf16(o[2 * dp], pa, b0, b1);
                mma_bf16(o[2 * dp + 1], pa, b2, b3);
            }
        }
        __syncthreads();
    }
    // normalise and store
#pragma unroll
    for (int h = 0; h < 2; h++) {
        float l = l_run[h];
        l += __shfl_xor_sync(0xffffffffu, l, 1);
        l += __shfl_xor_sync(0xffffffffu, l, 2);
        const float inv = 1.0f / l;
        const int r = warp * 16 + g + 8 * h;
        if (r < w.q_valid) {
            __nv_bfloat16* dst = ctx + (size_t)(w.q_row0 + r) * H + head * kD;
#pragma unroll
            for (int i = 0; i < 8; i++)
                *reinterpret_cast<uint32_t*>(dst + i * 8 + 2 * t) = pack2(o[i][2 * h] * inv, o[i][2 * h + 1] * inv);
        }
    }
}

}  // namespace

// enc::attention_f32_kernel lives in encoder_kernels.cuh (FP32 path); declared here for the dtype-0 branch
#include "encoder_kernels.cuh"

int attention_plan(anon_ctx* ctx, WsCursor& ws, const int32_t* h_cu, int B, int dtype, AttnPlan* plan)
{
    // h_cu points at this chunk's first sequence boundary; rows are relative to token h_cu[0]
    plan->d_work = nullptr; plan->n_items = 0;
    if (!ctx || !h_cu || B < 0) return ANON_ERR_INVALID_ARG;
    for (int s = 0; s < B; s++)
        if (h_cu[s + 1] < h_cu[s] || h_cu[s + 1] - h_cu[s] > 512) return ANON_ERR_UNSUPPORTED;
    if (dtype == 0 || B == 0) return ANON_OK;
    const int tok0 = h_cu[0];
    std::vector<WorkItem> items;
    items.reserve((size_t)(h_cu[B] - tok0) / kQT + B);
    for (int s = 0; s < B; s++) {
        const int a = h_cu[s] - tok0, n = h_cu[s + 1] - h_cu[s];
        for (int q0 = 0; q0 < n; q0 += kQT) items.push_back(WorkItem{a + q0, a, n, std::min(kQT, n - q0)});
    }
    if (items.empty()) return ANON_OK;
    std::stable_sort(items.begin(), items.end(), [](const WorkItem& x, const WorkItem& y) { return x.n > y.n; });
    const size_t bytes = items.size() * sizeof(WorkItem);
    void* d_work = ws.take(bytes);
    if (!d_work) return ANON_ERR_OOM;
    // pageable source: the runtime stages the bytes before cudaMemcpyAsync returns, so `items` may die
    CU_TRY(ctx, cudaMemcpyAsync(d_work, items.data(), bytes, cudaMemcpyHostToDevice, ctx->stream));
    plan->d_work = d_work; plan->n_items = (int)items.size();
    return ANON_OK;
}

int attention_run(anon_ctx* ctx, const AttnPlan& plan, const void* d_qkv, const int32_t* d_cu, int tok0, int B,
                  int hidden, int heads, int dtype, void* d_ctx)
{
    // d_qkv / d_ctx are chunk-local (row 0 = token tok0); d_cu points at the chunk's first sequence boundary
    if (!ctx || !d_qkv || !d_cu || !d_ctx) return ANON_ERR_INVALID_ARG;
    if (heads <= 0 || hidden != heads * 64) return ANON_ERR_UNSUPPORTED;
    if (B == 0) return ANON_OK;
    if (dtype == 0) {
        enc::attention_f32_kernel<<<dim3(B, heads), 128, 0, ctx->stream>>>((const float*)d_qkv, d_cu, 0, tok0, hidden, (float*)d_ctx);
        CU_LAUNCH_CHECK(ctx, "attention_f32_kernel");
        return ANON_OK;
    }
    if (plan.n_items == 0) return ANON_OK;
    attention_bf16_kernel<<<dim3((unsigned)plan.n_items, heads), 128, 0, ctx->stream>>>(
        (const __nv_bfloat16*)d_qkv, (const WorkItem*)plan.d_work, hidden, (__nv_bfloat16*)d_ctx);
    CU_LAUNCH_CHECK(ctx, "attention_bf16_kernel");
    return ANON_OK;
}

extern "C" int anon_attention(anon_ctx* ctx, const void* d_qkv, const int32_t* d_cu_seqlens, const int32_t* h_cu_seqlens,
                              int32_t B, int32_t T, int32_t hidden, int32_t heads, int32_t dtype, void* d_ctx)
{
    if (!ctx) return ANON_ERR_INVALID_ARG;
    CU_TRY(ctx, cudaSetDevice(ctx->device));
    if (!h_cu_seqlens || B < 0 || T < 0) return ANON_ERR_INVALID_ARG;
    WsCursor ws = ws_begin(ctx);
    AttnPlan plan;
    int rc = attention_plan(ctx, ws, h_cu_seqlens, B, dtype, &plan);
    if (rc) return rc;
    return attention_run(ctx, plan, d_qkv, d_cu_seqlens, h_cu_seqlens[0], B, hidden, heads, dtype, d_ctx);
}
