// gemm_tcgen05.cu -- K2: C[M,N] = A[M,K] * W[N,K]^T (+bias, +GELU | +residual) for the encoder's dense
// projections (S8a A2, A4, A5, A6; BJ "tcgen05/TMEM tensor-core GEMMs fed by TMA").
//
// sm_100a design: persistent CTA PAIRS (tcgen05 cta_group::2, one CTA per SM, clusters of 2): a pair computes a
// 256 x 256 tile, each CTA holding 128 accumulator rows in its TMEM and staging its 128 rows of A and only HALF of
// the B tile (the tensor cores of both SMs read both halves), which halves the shared-memory fill and operand
// traffic that capped the single-CTA version at ~70 % tensor-pipe activity.  Warp-specialised:
//   warp 0   TMA producer : (both CTAs) cp.async.bulk.tensor 2-D tiles (128B swizzle) of A [128 x 64] and W [128 x 64]
//                           into a 5-6 stage shared-memory ring; all bytes are counted on the LEADER's mbarrier
//   warp 1   MMA issuer   : one thread of the leader CTA issues tcgen05.mma.cta_group::2 (M=256, N=256, K=16,
//                           BF16 -> FP32) with shared-memory matrix descriptors; accumulators live in TMEM,
//                           double-buffered (2 x 256 columns) so the epilogue of tile i overlaps the mainloop of
//                           tile i+1; tcgen05.commit (multicast to both CTAs) frees ring slots / publishes accumulators
//   warp 2   TMEM allocator
//   warps 4-11 epilogue   : (both CTAs, two warps per TMEM lane quarter; 4 warps for the residual epilogue) tcgen05.ld (32 lanes x 32 columns per warp) -> bias / GELU / residual in registers
//                           -> 128B-swizzled shared-memory boxes (one row per thread, conflict-free) -> TMA store
//                           (coalesced, asynchronous, M/N tails clipped by the tensor map).  The FP32 residual
//                           tile arrives the same way: each epilogue warp TMA-loads its own 32x32 boxes three
//                           boxes ahead (also across tiles, so they land during the next mainloop), adds in
//                           place and stores from the same buffer.
// Outputs with N <= 128 use the single-CTA variant (CG = 1, 128 x 128 tiles).
// Operands are "TN": A row-major [M,K], W row-major [N,K] (both K-contiguous = K-major UMMA operands).
#include "common.cuh"
#include "ptx_sm100.cuh"

namespace {

constexpr int BM = 128;
constexpr int BK = 64;                    // 64 BF16 = 128 bytes = one swizzle row
constexpr int UMMA_K = 16;
constexpr int kThreads = 384;               // warps 0-3: TMA / MMA / TMEM alloc / idle; warps 4-11: epilogue
constexpr int A_STAGE_BYTES = BM * BK * 2;

// NB = FP32 residual boxes in flight per epilogue warp (EPI 2 only): 4 for short K (the epilogue's HBM traffic
// paces the kernel), 2 for long K (a fourth mainloop stage is worth more).
// CG = CTAs per MMA (tcgen05 cta_group): 1 = 128 x BN tile per CTA; 2 = a CTA pair computes 256 x BN, each CTA owning
// 128 rows of the accumulator and staging only half of the B tile (halves shared-memory fill and operand traffic).
constexpr int kRopeStride = 512;   // positions per pair row of the EPI 5 (cos, sin) table (max_pos <= 512)

template <int BN, int EPI, int NB, int CG, bool FOLD = false> struct Cfg {
    static constexpr int B_STAGE_BYTES = (BN / CG) * BK * 2;
    static constexpr int STAGE_BYTES = A_STAGE_BYTES + B_STAGE_BYTES;
    static constexpr int EPI_WARPS = (EPI == 2) ? 4 : 8;
    static constexpr int EPI_BYTES = (EPI == 2) ? 4 * NB * 4096 + 12288 + (FOLD ? 4 * 4096 : 0) /*FOLD: one BF16 box per warp*/ /*bias, gamma, beta staged for the epilogue*/ : 8 * 4096;   // 4 KB boxes
    static constexpr int STAGES = (227 * 1024 - 2048 - EPI_BYTES) / STAGE_BYTES > 6 ? 6 : (227 * 1024 - 2048 - EPI_BYTES) / STAGE_BYTES;
    static constexpr int TMEM_COLS = 2 * BN;                      // two accumulator buffers
    static constexpr int NUM_BARS = 2 * STAGES + 4 + 32;
    static constexpr int SMEM_BYTES = STAGES * STAGE_BYTES + EPI_BYTES + 1024 /*align slack*/ + 512 /*barriers*/;
};

__device__ __forceinline__ uint32_t pack_bf16(float a, float b);
// ---- packed FP32x2 arithmetic (sm_100 FFMA2 / FMUL2 / FADD2: two lanes per issue slot) ----
__device__ __forceinline__ uint64_t pk2(float a, float b) {
    uint64_t r; asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(a), "f"(b)); return r;
}
__device__ __forceinline__ void upk2(uint64_t v, float& a, float& b) { asm("mov.b64 {%0, %1}, %2;" : "=f"(a), "=f"(b) : "l"(v)); }
__device__ __forceinline__ uint64_t fma2(uint64_t a, uint64_t b, uint64_t c) {
    uint64_t d; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c)); return d;
}
__device__ __forceinline__ uint64_t mul2(uint64_t a, uint64_t b) {
    uint64_t d; asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b)); return d;
}
__device__ __forceinline__ uint64_t add2(uint64_t a, uint64_t b) {
    uint64_t d; asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b)); return d;
}
__device__ __forceinline__ float ex2_approx(float x) { float y; asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float rcp_approx(float x) { float y; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }

// erf-GELU (reading D3) for two values at once: gelu(z) = z * Phi(z) with Phi(z) = sigma(z * P(z^2)), P a degree-4
// polynomial in z^2 fitted (minimax, csrc/fit_gelu_coeffs.py) so that |z| * |sigma(z P(z^2)) - Phi(z)| <= 3.1e-6 for
// every z (the leading coefficient is positive, so the form saturates correctly and needs no clamp).  That is
// ~1e3 below the BF16 rounding of the stored activation.  The coefficients below carry the factor -log2(e) so that
// sigma(u) = 1 / (1 + 2^(u')).  Cost per pair: 8 packed FMA-pipe ops + 4 MUFU (ex2, rcp) + 1 convert.
__device__ __forceinline__ uint64_t gelu2_f32(uint64_t z) {
    constexpr float kL = -1.4426950408889634f;
    const uint64_t c1 = pk2(kL * 1.5956562720997576f, kL * 1.5956562720997576f);
    const uint64_t c3 = pk2(kL * 0.07293758090262617f, kL * 0.07293758090262617f);
    const uint64_t c5 = pk2(kL * -0.00024972250409287103f, kL * -0.00024972250409287103f);
    const uint64_t c7 = pk2(kL * -6.116217765511888e-05f, kL * -6.116217765511888e-05f);
    const uint64_t c9 = pk2(kL * 2.2381744780047116e-06f, kL * 2.2381744780047116e-06f);
    const uint64_t z2 = mul2(z, z);
    uint64_t p = fma2(c9, z2, c7);
    p = fma2(p, z2, c5);
    p = fma2(p, z2, c3);
    p = fma2(p, z2, c1);
    const uint64_t u = mul2(p, z);
    float u0, u1;
    upk2(u, u0, u1);
    const uint64_t e = pk2(ex2_approx(u0), ex2_approx(u1));
    const uint64_t d = add2(e, pk2(1.0f, 1.0f));
    float d0, d1;
    upk2(d, d0, d1);
    return mul2(z, pk2(rcp_approx(d0), rcp_approx(d1)));
}
__device__ __forceinline__ uint32_t gelu2_bf16(uint64_t z) {
    float g0, g1;
    upk2(gelu2_f32(z), g0, g1);
    return pack_bf16(g0, g1);
}

__device__ __forceinline__ uint32_t pack_bf16(float a, float b) {
    __nv_bfloat162 v = __floats2bfloat162_rn(a, b);
    return *reinterpret_cast<uint32_t*>(&v);
}
__device__ __forceinline__ void st_shared_v4(uint32_t addr, uint32_t a, uint32_t b, uint32_t c, uint32_t d) {
    asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(addr), "r"(a), "r"(b), "r"(c), "r"(d) : "memory");
}
__device__ __forceinline__ void ld_shared_2x2(uint32_t addr, uint64_t& lo, uint64_t& hi) {      // 4 floats as two FP32x2 pairs
    asm volatile("ld.shared.v2.b64 {%0, %1}, [%2];" : "=l"(lo), "=l"(hi) : "r"(addr) : "memory");
}
__device__ __forceinline__ void st_shared_2x2(uint32_t addr, uint64_t lo, uint64_t hi) {
    asm volatile("st.shared.v2.b64 [%0], {%1, %2};" ::"r"(addr), "l"(lo), "l"(hi) : "memory");
}
__device__ __forceinline__ float4 ld_shared_f4(uint32_t addr) {
    float4 v;
    asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(addr) : "memory");
    return v;
}

// EPI: 0 = +bias -> BF16;  1 = +bias, GELU -> BF16;  2 = +bias +residual(FP32) -> FP32;
//          (with res_stats: the residual is stored un-normalised and LayerNorm'ed on the fly, see gemm_bf16_res_ln_impl)
//      4 = GeGLU (NEXT-3): the tile's first BN/2 accumulator columns are a, the last BN/2 their gates (W's rows are
//          interleaved per tile by the caller); writes gelu(a) * gate as BF16 [M, N/2]; no bias
//      5 = QKV projection with rotary position embedding (NEXT-3): like 0 without bias; in the q and k column blocks
//          (columns < 2N/3) every 64-column box is one head and its pairs (j, j + 32) turn by the angle of the row's
//          position.  rope_tab = (cos, sin) table float2 [32][kRopeStride] (pair-major, so that the rows of a warp --
//          consecutive positions -- read consecutive entries), rope_pos = int position id per row
// FOLD (LayerNorm folded into the GEMMs; EPI 0 / 2 only): row statistics travel as PARTIAL sums, part[row][i] = (sum, sum of
// squares) over the 256 columns of n-tile i of the GEMM that produced the row, stat_cnt = H / 256 of them, summed in a fixed
// order (deterministic, no atomics); mean = S / H, rstd = 1 / sqrt(Q / H - mean^2 + eps).
//   EPI 2 + FOLD (producer): besides C = acc + bias + LN(residual) as FP32 it writes bf16(C) through tmap_yb (the NEXT GEMM's
//          raw A operand) and part_out[row][n_blk]; the residual's own (mean, rstd) come from part_in instead of res_stats.
//   EPI 0 + FOLD (consumer): A holds raw rows y, W holds bf16(W * gamma); the epilogue finishes the LayerNorm:
//          z = rstd * (acc - mean * s_n) + c_n with fold_s[n] = sum_k W'[n,k] and bias[n] = c_n = b_n + sum_k beta_k W[n,k].
__device__ __forceinline__ float2 row_stats_from_partials(const float2* __restrict__ part, int row, int cnt, float inv_h, float eps) {
    float s = 0.f, q = 0.f;
    for (int i = 0; i < cnt; i++) { const float2 p = __ldg(part + (size_t)row * cnt + i); s += p.x; q += p.y; }
    const float mean = s * inv_h;
    const float var = fmaxf(q * inv_h - mean * mean, 0.f);
    return make_float2(mean, 1.0f / sqrtf(var + eps));
}

template <int BN, int EPI, int NB, int CG, bool FOLD>
__global__ void __launch_bounds__(kThreads, 1)
gemm_bf16_tcgen05_kernel(const __grid_constant__ CUtensorMap tmap_a, const __grid_constant__ CUtensorMap tmap_b,
                         const __grid_constant__ CUtensorMap tmap_c, const __grid_constant__ CUtensorMap tmap_r,
                         const __grid_constant__ CUtensorMap tmap_yb,
                         const float* __restrict__ bias, const float* __restrict__ ln_g, const float* __restrict__ ln_b,
                         const float2* __restrict__ res_stats, const float2* __restrict__ rope_tab,
                         const int* __restrict__ rope_pos, const float2* __restrict__ part_in, int stat_cnt, float inv_h, float ln_eps,
                         float2* __restrict__ part_out, const float* __restrict__ fold_s, int M, int N, int K)
{
    static_assert(!FOLD || EPI == 0 || EPI == 2, "FOLD: the plain (consumer) and the residual (producer) epilogue only");
    using C = Cfg<BN, EPI, NB, CG, FOLD>;
    extern __shared__ uint8_t smem_raw[];
    const uint32_t smem_base = (ptx::smem_u32(smem_raw) + 1023u) & ~1023u;
    const uint32_t epi_base = smem_base + C::STAGES * C::STAGE_BYTES;
    const uint32_t bar_base = epi_base + C::EPI_BYTES;
    auto full_bar = [&](int s) { return bar_base + 8u * s; };
    auto empty_bar = [&](int s) { return bar_base + 8u * (C::STAGES + s); };
    auto tfull_bar = [&](int a) { return bar_base + 8u * (2 * C::STAGES + a); };
    auto tempty_bar = [&](int a) { return bar_base + 8u * (2 * C::STAGES + 2 + a); };
    auto rfull_bar = [&](int q, int b) { return bar_base + 8u * (2 * C::STAGES + 4 + 8 * q + b); };      // up to 8 boxes per warp
    const uint32_t tmem_slot = bar_base + 8u * C::NUM_BARS;
    uint32_t* tmem_slot_ptr = reinterpret_cast<uint32_t*>(smem_raw + (tmem_slot - ptx::smem_u32(smem_raw)));

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int rank = CG == 2 ? (int)ptx::cluster_ctarank() : 0;          // position in the CTA pair; 0 issues the MMAs
    const int cid = (int)blockIdx.x / CG, ncl = (int)gridDim.x / CG;     // tile scheduler works on pairs
    constexpr int TM = BM * CG;                                         // rows per tile
    const int num_m = (M + TM - 1) / TM, num_n = (N + BN - 1) / BN;
    const int num_tiles = num_m * num_n;
    const int num_kb = K / BK;
    // local tile lt of this CTA (pair) -> (m_blk, n_blk)
    auto get_tile = [&](int lt, int& m_blk, int& n_blk) -> bool {
        if ((EPI <= 1 || EPI >= 4) && num_m >= 2 * ncl) {
            // short-K GEMMs with many row blocks: a pair keeps its row block of A (256 x K, L2-resident across the
            // pairs) for all n-tiles, starting at a different n so that the pairs do not ask for the same W tile at once
            m_blk = cid + (lt / num_n) * ncl; n_blk = (lt + cid) % num_n; return m_blk < num_m;
        }
        const int tile = cid + lt * ncl;
        m_blk = tile / num_n; n_blk = tile % num_n;
        return tile < num_tiles;
    };

    if (warp == 0 && lane == 0) {
        ptx::prefetch_tensormap(&tmap_a);
        ptx::prefetch_tensormap(&tmap_b);
        ptx::prefetch_tensormap(&tmap_c);
        if (EPI >= 2) ptx::prefetch_tensormap(&tmap_r);
        if (EPI == 2 && FOLD) ptx::prefetch_tensormap(&tmap_yb);
    }
    if (warp == 1 && lane == 0) {
        for (int s = 0; s < C::STAGES; s++) { ptx::mbar_init(full_bar(s), 1); ptx::mbar_init(empty_bar(s), 1); }
        for (int a = 0; a < 2; a++) { ptx::mbar_init(tfull_bar(a), 1); ptx::mbar_init(tempty_bar(a), CG * C::EPI_WARPS); }
        for (int i = 0; i < 32; i++) ptx::mbar_init(rfull_bar(i >> 3, i & 7), 1);
        ptx::fence_barrier_init();
        ptx::fence_proxy_async();
    }
    if constexpr (EPI == 2) {             // bias (and gamma / beta of the residual's LayerNorm) -> shared memory: every
        if (N <= 1024) {                  // epilogue thread reads all N of them per row
            float* par = reinterpret_cast<float*>(smem_raw + (epi_base + 4 * NB * 4096 - ptx::smem_u32(smem_raw)));
            for (int i = threadIdx.x; i < N; i += kThreads) {
                par[i] = bias[i];
                par[1024 + i] = (res_stats || (FOLD && part_in)) ? ln_g[i] : 1.f;
                par[2048 + i] = (res_stats || (FOLD && part_in)) ? ln_b[i] : 0.f;
            }
        }
    }
    if (warp == 2) {
        if (CG == 2) { ptx::tmem_alloc_cg2(tmem_slot, C::TMEM_COLS); ptx::tmem_relinquish_cg2(); }
        else { ptx::tmem_alloc(tmem_slot, C::TMEM_COLS); ptx::tmem_relinquish(); }
    }
    ptx::tc_fence_before();
    if (CG == 2) ptx::cluster_sync(); else __syncthreads();            // the peer's barriers must be initialised too
    ptx::tc_fence_after();
    const uint32_t tmem_base = *tmem_slot_ptr;

    if (warp == 0) {
        // ===== TMA producer (one per CTA): A rows [rank*128, +128) of the tile, B rows [rank*BN/CG, +BN/CG) =====
        if (lane == 0) {
            int s = 0; uint32_t ph = 0;
            int m_blk, n_blk;
            for (int lt = 0; get_tile(lt, m_blk, n_blk); lt++) {
                for (int kb = 0; kb < num_kb; kb++) {
                    ptx::mbar_wait_backoff(empty_bar(s), ph ^ 1u);
                    const uint32_t sa = smem_base + s * C::STAGE_BYTES;
                    if (CG == 1) {
                        ptx::mbar_arrive_expect_tx(full_bar(s), C::STAGE_BYTES);
                        ptx::tma_load_2d(sa, &tmap_a, full_bar(s), kb * BK, m_blk * BM);
                        ptx::tma_load_2d(sa + A_STAGE_BYTES, &tmap_b, full_bar(s), kb * BK, n_blk * BN);
                    } else {
                        // both CTAs' bytes are counted on the LEADER's barrier (it alone waits before issuing the MMA); only
                        // the leader arrives.  The peer cannot run a phase ahead: its empty barrier of this stage fires
                        // after the MMAs that the leader issued on the previous phase of the same full barrier.
                        const uint32_t lead_full = ptx::mapa(full_bar(s), 0);
                        if (rank == 0) ptx::mbar_arrive_expect_tx(full_bar(s), 2 * C::STAGE_BYTES);
                        ptx::tma_load_2d_cg2(sa, &tmap_a, lead_full, kb * BK, m_blk * TM + rank * BM);
                        ptx::tma_load_2d_cg2(sa + A_STAGE_BYTES, &tmap_b, lead_full, kb * BK, n_blk * BN + rank * (BN / CG));
                    }
                    if (++s == C::STAGES) { s = 0; ph ^= 1u; }
                }
            }
        }
    } else if (warp == 1) {
        // ===== MMA issuer: one thread of the leader CTA =====
        if (lane == 0 && rank == 0) {
            constexpr uint32_t idesc = ptx::make_idesc_bf16(TM, BN);
            int s = 0; uint32_t ph = 0;
            int acc = 0; uint32_t acc_ph = 0;
            int m_blk, n_blk;
            for (int lt = 0; get_tile(lt, m_blk, n_blk); lt++) {
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
                        if (CG == 2) ptx::mma_f16_ss_cg2(d_tmem, adesc + (uint64_t)(2 * k), bdesc + (uint64_t)(2 * k), idesc, (kb | k) ? 1u : 0u);
                        else ptx::mma_f16_ss(d_tmem, adesc + (uint64_t)(2 * k), bdesc + (uint64_t)(2 * k), idesc, (kb | k) ? 1u : 0u);
                    }
                    if (CG == 2) ptx::mma_commit_cg2(empty_bar(s)); else ptx::mma_commit(empty_bar(s));
                    if (++s == C::STAGES) { s = 0; ph ^= 1u; }
                }
                if (CG == 2) ptx::mma_commit_cg2(tfull_bar(acc)); else ptx::mma_commit(tfull_bar(acc));
                if (++acc == 2) { acc = 0; acc_ph ^= 1u; }
            }
        }
    } else if (warp >= 4 && warp < 4 + C::EPI_WARPS) {
        const int q = warp & 3;                       // TMEM lane quarter this warp may access
        const uint32_t row_off = (uint32_t)lane * 128u;      // this thread's row inside a 32-row box
        const uint32_t sw = (uint32_t)(lane & 7);            // 128B swizzle: 16-byte chunk index ^= row & 7
        auto arrive_tempty = [&](int a) {               // the accumulator is handed back to the LEADER's MMA thread
            if (CG == 2) ptx::mbar_arrive_cluster(ptx::mapa(tempty_bar(a), 0)); else ptx::mbar_arrive(tempty_bar(a));
        };
        int acc = 0; uint32_t acc_ph = 0;
        uint32_t nbox = 0;                            // boxes this warp has handled (buffer ring position)
        (void)nbox;

        if constexpr (EPI == 2) {
            constexpr int BPT = BN / 32;              // 32x32 FP32 boxes per tile per warp
            const uint32_t stg = epi_base + (uint32_t)(q * NB * 4096);
            const uint32_t par_base = epi_base + 4u * NB * 4096u;      // gamma | beta, 1024 floats each
            uint32_t rph = 0;                         // phase bit of each residual buffer's barrier
            auto issue_load = [&](uint32_t i) {       // lane 0: residual box i -> buffer i % NB
                int mb, nb;
                if (!get_tile((int)(i / BPT), mb, nb)) return;
                const int row0 = mb * TM + rank * BM + q * 32, col = nb * BN + (int)(i % BPT) * 32;
                if (row0 >= M || col >= N) return;
                const uint32_t bar = rfull_bar(q, i % NB);
                ptx::mbar_arrive_expect_tx(bar, 4096);
                ptx::tma_load_2d(stg + (i % NB) * 4096u, &tmap_r, bar, col, row0);
            };
            if (lane == 0) { for (uint32_t i = 0; i + 1 < NB; i++) issue_load(i); }
            int m_blk, n_blk;
            const uint32_t xbuf = epi_base + 4u * NB * 4096u + 12288u + (uint32_t)(q * 4096);   // FOLD: this warp's BF16 box (32 rows x 64 columns)
            (void)xbuf;
            const bool res_ln = res_stats != nullptr || (FOLD && part_in != nullptr);      // the residual needs its LayerNorm
            auto load_stats = [&](int rn) -> float2 {
                if (FOLD && part_in) return row_stats_from_partials(part_in, rn, stat_cnt, inv_h, ln_eps);
                return __ldg(res_stats + rn);
            };
            float2 st_next = make_float2(0.f, 1.f);
            if (res_ln && get_tile(0, m_blk, n_blk)) {
                const int rn = m_blk * TM + rank * BM + q * 32 + lane;
                if (rn < M) st_next = load_stats(rn);
            }
            float f_sum = 0.f, f_sq = 0.f;            // FOLD: this row's partial statistics over the tile's columns
            for (int lt = 0; get_tile(lt, m_blk, n_blk); lt++) {
                const int row0 = m_blk * TM + rank * BM + q * 32;
                // (mean, rstd) of this thread's residual row: loaded one tile ahead so that no box waits for it
                const float r_mu = st_next.x, r_rs = st_next.y;
                {
                    int mb2, nb2;
                    if (res_ln && get_tile(lt + 1, mb2, nb2)) {
                        const int rn = mb2 * TM + rank * BM + q * 32 + lane;
                        if (rn < M) st_next = load_stats(rn);
                    }
                }
                ptx::mbar_wait(tfull_bar(acc), acc_ph);
                ptx::tc_fence_after();
                const uint32_t t_base = tmem_base + ((uint32_t)(q * 32) << 16) + (uint32_t)(acc * BN);
#pragma unroll 1
                for (int j = 0; j < BPT; j++, nbox++) {
                    const int col = n_blk * BN + j * 32;
                    const uint32_t b = nbox % NB;
                    const uint32_t buf = stg + b * 4096u;
                    uint32_t r[32];
                    ptx::tmem_ld_32x32b_x32(t_base + (uint32_t)(j * 32), r);
                    ptx::tmem_ld_wait();
                    if (j == BPT - 1) {               // accumulator fully read: hand it back to the MMA warp
                        ptx::tc_fence_before();
                        __syncwarp();
                        if (lane == 0) arrive_tempty(acc);
                    }
                    const bool valid = row0 < M && col < N;      // warp-uniform
                    if (valid) {
                        ptx::mbar_wait(rfull_bar(q, b), (rph >> b) & 1u);
                        rph ^= 1u << b;
                        if (N <= 1024) {              // parameters from shared memory, packed FP32x2 arithmetic
                            const uint64_t rs2 = pk2(r_rs, r_rs), nmr2 = pk2(-r_mu * r_rs, -r_mu * r_rs);
#pragma unroll
                            for (int v = 0; v < 8; v++) {
                                const uint32_t addr = buf + row_off + (((uint32_t)v ^ sw) << 4);
                                const uint32_t pc = par_base + (uint32_t)(col + 4 * v) * 4u;
                                uint64_t x0, x1, b0, b1;
                                ld_shared_2x2(addr, x0, x1);
                                ld_shared_2x2(pc, b0, b1);
                                if (res_ln) {             // the residual is stored un-normalised: x = LN(y) on the fly
                                    uint64_t g0, g1, e0, e1;
                                    ld_shared_2x2(pc + 4096u, g0, g1);
                                    ld_shared_2x2(pc + 8192u, e0, e1);
                                    x0 = fma2(fma2(x0, rs2, nmr2), g0, e0);
                                    x1 = fma2(fma2(x1, rs2, nmr2), g1, e1);
                                }
                                const uint64_t o01 = add2(add2(pk2(__uint_as_float(r[4 * v + 0]), __uint_as_float(r[4 * v + 1])), b0), x0);
                                const uint64_t o23 = add2(add2(pk2(__uint_as_float(r[4 * v + 2]), __uint_as_float(r[4 * v + 3])), b1), x1);
                                st_shared_2x2(addr, o01, o23);
                                if (FOLD) {               // keep the values for the statistics and the BF16 copy (r[] is free now)
                                    float o0, o1, o2, o3;
                                    upk2(o01, o0, o1); upk2(o23, o2, o3);
                                    r[4 * v + 0] = __float_as_uint(o0); r[4 * v + 1] = __float_as_uint(o1);
                                    r[4 * v + 2] = __float_as_uint(o2); r[4 * v + 3] = __float_as_uint(o3);
                                }
                            }
                            if (FOLD) {
                                if (j == 0) { f_sum = 0.f; f_sq = 0.f; }
                                uint64_t s2a = pk2(0.f, 0.f), s2b = s2a, q2a = s2a, q2b = s2a;      // packed FP32x2 partial sums
#pragma unroll
                                for (int e = 0; e < 32; e += 4) {
                                    const uint64_t v01 = pk2(__uint_as_float(r[e]), __uint_as_float(r[e + 1]));
                                    const uint64_t v23 = pk2(__uint_as_float(r[e + 2]), __uint_as_float(r[e + 3]));
                                    s2a = add2(s2a, v01); s2b = add2(s2b, v23);
                                    q2a = fma2(v01, v01, q2a); q2b = fma2(v23, v23, q2b);
                                }
                                float sa, sb, qa, qb;
                                upk2(add2(s2a, s2b), sa, sb); upk2(add2(q2a, q2b), qa, qb);
                                f_sum += sa + sb;
                                f_sq += qa + qb;
                                if (!(j & 1)) {           // the BF16 box is refilled: its store (committed BEFORE the FP32 store of the
                                    if (lane == 0) ptx::bulk_wait_read<1>();      // same iteration, see below) must have read it; the newest
                                    __syncwarp();                                 // group -- that FP32 store -- may still be in flight
                                }
#pragma unroll
                                for (int c4 = 0; c4 < 4; c4++)      // 16-byte chunks (j & 1) * 4 + c4 of the 64-column BF16 row
                                    st_shared_v4(xbuf + row_off + ((((uint32_t)((j & 1) * 4 + c4)) ^ sw) << 4),
                                                 pack_bf16(__uint_as_float(r[8 * c4 + 0]), __uint_as_float(r[8 * c4 + 1])),
                                                 pack_bf16(__uint_as_float(r[8 * c4 + 2]), __uint_as_float(r[8 * c4 + 3])),
                                                 pack_bf16(__uint_as_float(r[8 * c4 + 4]), __uint_as_float(r[8 * c4 + 5])),
                                                 pack_bf16(__uint_as_float(r[8 * c4 + 6]), __uint_as_float(r[8 * c4 + 7])));
                                if (j == BPT - 1 && row0 + lane < M) part_out[(size_t)(row0 + lane) * num_n + n_blk] = make_float2(f_sum, f_sq);
                            }
                        } else {
#pragma unroll
                            for (int v = 0; v < 8; v++) {
                                const uint32_t addr = buf + row_off + (((uint32_t)v ^ sw) << 4);
                                const float4 x = ld_shared_f4(addr);
                                float4 bb = make_float4(0.f, 0.f, 0.f, 0.f);
                                if (col + 4 * v < N) bb = __ldg(reinterpret_cast<const float4*>(bias + col + 4 * v));
                                st_shared_v4(addr, __float_as_uint(__uint_as_float(r[4 * v + 0]) + bb.x + x.x),
                                             __float_as_uint(__uint_as_float(r[4 * v + 1]) + bb.y + x.y),
                                             __float_as_uint(__uint_as_float(r[4 * v + 2]) + bb.z + x.z),
                                             __float_as_uint(__uint_as_float(r[4 * v + 3]) + bb.w + x.w));
                            }
                        }
                        ptx::fence_proxy_async();
                        __syncwarp();
                        if (lane == 0) {
                            if (FOLD && (j & 1)) {        // a bulk group of its own, OLDER than this iteration's FP32 store
                                ptx::tma_store_2d(&tmap_yb, xbuf, col - 32, row0);
                                ptx::bulk_commit();
                            }
                            ptx::tma_store_2d(&tmap_c, buf, col, row0);
                        }
                    }
                    if (lane == 0) {
                        ptx::bulk_commit();
                        ptx::bulk_wait_read<1>();     // the store of box nbox-1 has read its buffer: refill it
                        issue_load(nbox + NB - 1);
                    }
                    __syncwarp();
                }
                if (++acc == 2) { acc = 0; acc_ph ^= 1u; }
            }
        } else {
            // two warps per TMEM lane quarter, each owning half of the tile's columns and one 4 KB staging box
            const int half = (warp - 4) >> 2;
            const uint32_t buf = epi_base + (uint32_t)((warp - 4) * 4096);
            int m_blk, n_blk;
            uint64_t fa2 = 0, fb2 = 0;
            int fold_mblk = -1;
            (void)fa2; (void)fb2; (void)fold_mblk;
            for (int lt = 0; get_tile(lt, m_blk, n_blk); lt++) {
                const int row0 = m_blk * TM + rank * BM + q * 32;
                // FOLD consumer: z = a * acc + (b * s_n + c_n) with a = rstd, b = -rstd * mean of this thread's (raw) A row
                if (FOLD && m_blk != fold_mblk) {         // the pair keeps a row block for all its n-tiles: one load per row block
                    float2 st = make_float2(0.f, 1.f);
                    if (row0 + lane < M) st = row_stats_from_partials(part_in, row0 + lane, stat_cnt, inv_h, ln_eps);
                    fa2 = pk2(st.y, st.y); fb2 = pk2(-st.x * st.y, -st.x * st.y);
                    fold_mblk = m_blk;
                }
                ptx::mbar_wait(tfull_bar(acc), acc_ph);
                ptx::tc_fence_after();
                const uint32_t t_base = tmem_base + ((uint32_t)(q * 32) << 16) + (uint32_t)(acc * BN);
                if constexpr (EPI == 4) {
                    // this warp's 64 output columns: a = accumulator columns [half*64, +64), gates = [BN/2 + half*64, +64)
                    static_assert(EPI != 4 || BN == 256, "GeGLU epilogue: 256-column tiles");
                    const int col = n_blk * (BN / 2) + half * 64;
                    uint32_t o[32];
#pragma unroll
                    for (int hh = 0; hh < 2; hh++) {
                        uint32_t ra[32], rg[32];
                        ptx::tmem_ld_32x32b_x32(t_base + (uint32_t)(half * 64 + hh * 32), ra);
                        ptx::tmem_ld_32x32b_x32(t_base + (uint32_t)(BN / 2 + half * 64 + hh * 32), rg);
                        ptx::tmem_ld_wait();
                        if (hh == 1) {                             // this warp's share of the accumulator is read
                            ptx::tc_fence_before();
                            __syncwarp();
                            if (lane == 0) arrive_tempty(acc);
                        }
#pragma unroll
                        for (int v = 0; v < 8; v++) {
                            float a0, a1, a2, a3;
                            upk2(mul2(gelu2_f32(pk2(__uint_as_float(ra[4 * v]), __uint_as_float(ra[4 * v + 1]))),
                                      pk2(__uint_as_float(rg[4 * v]), __uint_as_float(rg[4 * v + 1]))), a0, a1);
                            upk2(mul2(gelu2_f32(pk2(__uint_as_float(ra[4 * v + 2]), __uint_as_float(ra[4 * v + 3]))),
                                      pk2(__uint_as_float(rg[4 * v + 2]), __uint_as_float(rg[4 * v + 3]))), a2, a3);
                            o[hh * 16 + 2 * v] = pack_bf16(a0, a1);
                            o[hh * 16 + 2 * v + 1] = pack_bf16(a2, a3);
                        }
                    }
                    if (row0 < M && col < N / 2) {                 // warp-uniform
                        if (lane == 0) ptx::bulk_wait_read<0>();   // the previous store has read the staging box
                        __syncwarp();
#pragma unroll
                        for (int v = 0; v < 8; v++)
                            st_shared_v4(buf + row_off + (((uint32_t)v ^ sw) << 4), o[4 * v], o[4 * v + 1], o[4 * v + 2], o[4 * v + 3]);
                        ptx::fence_proxy_async();
                        __syncwarp();
                        if (lane == 0) { ptx::tma_store_2d(&tmap_c, buf, col, row0); ptx::bulk_commit(); }
                    }
                } else {
#pragma unroll 1
                for (int c0 = half * (BN / 2); c0 < (half + 1) * (BN / 2); c0 += 64) {   // 32-row x 64-column BF16 boxes
                    const int col = n_blk * BN + c0;
                    uint32_t r[64];
                    ptx::tmem_ld_32x32b_x32(t_base + (uint32_t)c0, r);
                    ptx::tmem_ld_32x32b_x32(t_base + (uint32_t)(c0 + 32), r + 32);
                    ptx::tmem_ld_wait();
                    if (c0 + 64 == (half + 1) * (BN / 2)) {       // this warp's share of the accumulator is read
                        ptx::tc_fence_before();
                        __syncwarp();
                        if (lane == 0) arrive_tempty(acc);
                    }
                    if (EPI == 5 && row0 < M && col < 2 * (N / 3)) {   // warp-uniform: a q or k head
                        const int row = row0 + lane;
                        const int p = row < M ? rope_pos[row] : 0;
                        const float2* tab = rope_tab + p;
#pragma unroll
                        for (int j = 0; j < 32; j++) {
                            const float2 cs = __ldg(tab + j * kRopeStride);
                            const float a = __uint_as_float(r[j]), b = __uint_as_float(r[j + 32]);
                            r[j] = __float_as_uint(a * cs.x - b * cs.y);
                            r[j + 32] = __float_as_uint(b * cs.x + a * cs.y);
                        }
                    }
                    if (row0 < M && col < N) {                     // warp-uniform
                        uint32_t o[32];
#pragma unroll
                        for (int v = 0; v < 16; v++) {             // 4 columns per step; N % 8 == 0
                            float4 bb = make_float4(0.f, 0.f, 0.f, 0.f);
                            if (EPI != 5 && col + 4 * v < N) bb = __ldg(reinterpret_cast<const float4*>(bias + col + 4 * v));
                            uint64_t z0, z1;
                            if (FOLD) {
                                float4 ss = make_float4(0.f, 0.f, 0.f, 0.f);
                                if (col + 4 * v < N) ss = __ldg(reinterpret_cast<const float4*>(fold_s + col + 4 * v));
                                z0 = fma2(pk2(__uint_as_float(r[4 * v + 0]), __uint_as_float(r[4 * v + 1])), fa2, fma2(fb2, pk2(ss.x, ss.y), pk2(bb.x, bb.y)));
                                z1 = fma2(pk2(__uint_as_float(r[4 * v + 2]), __uint_as_float(r[4 * v + 3])), fa2, fma2(fb2, pk2(ss.z, ss.w), pk2(bb.z, bb.w)));
                            } else {
                                z0 = add2(pk2(__uint_as_float(r[4 * v + 0]), __uint_as_float(r[4 * v + 1])), pk2(bb.x, bb.y));
                                z1 = add2(pk2(__uint_as_float(r[4 * v + 2]), __uint_as_float(r[4 * v + 3])), pk2(bb.z, bb.w));
                            }
                            if (EPI == 1) {
                                o[2 * v] = gelu2_bf16(z0);
                                o[2 * v + 1] = gelu2_bf16(z1);
                            } else {
                                float a0, a1, a2, a3;
                                upk2(z0, a0, a1); upk2(z1, a2, a3);
                                o[2 * v] = pack_bf16(a0, a1);
                                o[2 * v + 1] = pack_bf16(a2, a3);
                            }
                        }
                        if (lane == 0) ptx::bulk_wait_read<0>();   // the previous store has read the staging box
                        __syncwarp();
#pragma unroll
                        for (int v = 0; v < 8; v++)
                            st_shared_v4(buf + row_off + (((uint32_t)v ^ sw) << 4), o[4 * v], o[4 * v + 1], o[4 * v + 2], o[4 * v + 3]);
                        ptx::fence_proxy_async();
                        __syncwarp();
                        if (lane == 0) { ptx::tma_store_2d(&tmap_c, buf, col, row0); ptx::bulk_commit(); }
                    }
                }
                }
                if (++acc == 2) { acc = 0; acc_ph ^= 1u; }
            }
        }
        if (lane == 0) ptx::bulk_wait<0>();           // every store has completed before shared memory goes away
    }

    ptx::tc_fence_before();
    if (CG == 2) ptx::cluster_sync(); else __syncthreads();            // no CTA of a pair leaves while its peer may still signal it
    if (warp == 2) {
        ptx::tc_fence_after();
        if (CG == 2) ptx::tmem_dealloc_cg2(tmem_base, C::TMEM_COLS); else ptx::tmem_dealloc(tmem_base, C::TMEM_COLS);
    }
}

}  // namespace

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

// 2-D row-major tensor [rows, cols] of `esize`-byte elements, box [box_rows, box_cols] (box_cols * esize = 128 B),
// 128-byte swizzle.
int make_tmap_2d(anon_ctx* ctx, CUtensorMap* tm, CUtensorMapDataType dt, uint32_t esize, const void* base, uint64_t rows,
                 uint64_t cols, uint32_t box_cols, uint32_t box_rows) {
    if (!ctx->encode_tiled) {
        void* fn = nullptr;
        cudaDriverEntryPointQueryResult q;
        cudaError_t e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &q);
        if (e != cudaSuccess || q != cudaDriverEntryPointSuccess || !fn)
            return cuda_fail(ctx, e == cudaSuccess ? cudaErrorUnknown : e, "cudaGetDriverEntryPoint(cuTensorMapEncodeTiled)");
        ctx->encode_tiled = fn;
    }
    for (size_t i = 0; i < ctx->tmap_keys.size(); i++) {
        const anon_ctx::TmapKey& k = ctx->tmap_keys[i];
        if (k.base == base && k.rows == rows && k.cols == cols && k.box_cols == box_cols && k.box_rows == box_rows && k.dt == (uint32_t)dt) {
            *tm = ctx->tmap_vals[i];
            return ANON_OK;
        }
    }
    const cuuint64_t gdim[2] = {cols, rows};
    const cuuint64_t gstride[1] = {cols * esize};
    const cuuint32_t box[2] = {box_cols, box_rows};
    const cuuint32_t estr[2] = {1, 1};
    CUresult r = ((EncodeTiledFn)ctx->encode_tiled)(tm, dt, 2, const_cast<void*>(base), gdim, gstride, box, estr,
                                                    CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
                                                    CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) {
        snprintf(ctx->cuda_err, sizeof ctx->cuda_err, "cuTensorMapEncodeTiled failed: CUresult %d", (int)r);
        return ANON_ERR_CUDA;
    }
    if (ctx->tmap_keys.size() >= 512) { ctx->tmap_keys.clear(); ctx->tmap_vals.clear(); }     // bounded: start over
    ctx->tmap_keys.push_back(anon_ctx::TmapKey{base, rows, cols, box_cols, box_rows, (uint32_t)dt});
    ctx->tmap_vals.push_back(*tm);
    return ANON_OK;
}

namespace {

struct LnArgs { const float* gamma = nullptr; const float* beta = nullptr; const float2* res_stats = nullptr;
                const float2* rope_tab = nullptr; const int* rope_pos = nullptr;
                // FOLD
                const float2* part_in = nullptr; int stat_cnt = 0; int stat_cols = 1; float eps = 0.f;
                float2* part_out = nullptr; void* yb_out = nullptr; const float* fold_s = nullptr; };

template <int BN, int EPI, int NB, int CG, bool FOLD = false>
int launch_gemm(anon_ctx* ctx, const __nv_bfloat16* A, const __nv_bfloat16* W, const float* bias, const float* residual,
                void* Cout, int M, int N, int K, const LnArgs* ln = nullptr)
{
    using C = Cfg<BN, EPI, NB, CG, FOLD>;
    const int tiles = ((M + BM * CG - 1) / (BM * CG)) * ((N + BN - 1) / BN);
    const int slots = ctx->sm_count / CG;
    int grid = CG * (tiles < slots ? tiles : slots);
    CUtensorMap ta, tb, tc, tr, tyb;
    int rc = make_tmap_2d(ctx, &ta, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, A, (uint64_t)M, (uint64_t)K, BK, BM);
    if (rc) return rc;
    rc = make_tmap_2d(ctx, &tb, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, W, (uint64_t)N, (uint64_t)K, BK, BN / CG);
    if (rc) return rc;
    if (EPI == 2) {
        rc = make_tmap_2d(ctx, &tc, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 4, Cout, (uint64_t)M, (uint64_t)N, 32, 32);
        if (rc) return rc;
        rc = make_tmap_2d(ctx, &tr, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 4, residual, (uint64_t)M, (uint64_t)N, 32, 32);
        if (rc) return rc;
    } else {
        rc = make_tmap_2d(ctx, &tc, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, Cout, (uint64_t)M, (uint64_t)(EPI == 4 ? N / 2 : N), 64, 32);
        if (rc) return rc;
        tr = tc;
    }
    tyb = tc;
    if (EPI == 2 && FOLD) {
        rc = make_tmap_2d(ctx, &tyb, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, ln->yb_out, (uint64_t)M, (uint64_t)N, 64, 32);
        if (rc) return rc;
    }
    auto kern = gemm_bf16_tcgen05_kernel<BN, EPI, NB, CG, FOLD>;
    rc = ensure_smem_attr(ctx, (const void*)kern, C::SMEM_BYTES);
    if (rc) return rc;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)grid); cfg.blockDim = dim3(kThreads); cfg.dynamicSmemBytes = C::SMEM_BYTES; cfg.stream = ctx->stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = CG; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr; cfg.numAttrs = 1;
    const float* g = ln ? ln->gamma : nullptr;
    const float* be = ln ? ln->beta : nullptr;
    const float2* rs = ln ? ln->res_stats : nullptr;
    const float2* rtab = ln ? ln->rope_tab : nullptr;
    const int* rpos = ln ? ln->rope_pos : nullptr;
    const float2* pin = ln ? ln->part_in : nullptr;
    const int scnt = ln ? ln->stat_cnt : 0;
    const float inv_h = ln ? 1.0f / (float)ln->stat_cols : 1.f;
    const float eps = ln ? ln->eps : 0.f;
    float2* pout = ln ? ln->part_out : nullptr;
    const float* fs = ln ? ln->fold_s : nullptr;
    CU_TRY(ctx, cudaLaunchKernelEx(&cfg, kern, ta, tb, tc, tr, tyb, bias, g, be, rs, rtab, rpos, pin, scnt, inv_h, eps, pout, fs, M, N, K));
    CU_LAUNCH_CHECK(ctx, "gemm_bf16_tcgen05_kernel");
    return ANON_OK;
}

}  // namespace

int gemm_bf16_impl(anon_ctx* ctx, const __nv_bfloat16* A, const __nv_bfloat16* W, const float* bias,
                   const float* residual, void* Cout, int M, int N, int K, int epilogue)
{
    if (!ctx || !A || !W || !bias || !Cout || M < 0 || N <= 0 || K <= 0 || epilogue < 0 || epilogue == 3 || epilogue > 4 ||
        (epilogue == 2 && !residual))
        return ANON_ERR_INVALID_ARG;
    if (K % BK != 0 || N % 8 != 0) return ANON_ERR_UNSUPPORTED;
    if (epilogue == 4 && N % 256 != 0) return ANON_ERR_UNSUPPORTED;       // whole (a | gate) tiles only
    if (M == 0) return ANON_OK;
    if (epilogue == 4) return launch_gemm<256, 4, 2, 2>(ctx, A, W, bias, residual, Cout, M, N, K);
    const bool long_k = K >= 2048;
    if (N > 128) {                 // CTA pairs: 256 x 256 tiles
        switch (epilogue) {
            case 0: return launch_gemm<256, 0, 2, 2>(ctx, A, W, bias, residual, Cout, M, N, K);
            case 1: return launch_gemm<256, 1, 2, 2>(ctx, A, W, bias, residual, Cout, M, N, K);
            default: return long_k ? launch_gemm<256, 2, 2, 2>(ctx, A, W, bias, residual, Cout, M, N, K)
                                   : launch_gemm<256, 2, 4, 2>(ctx, A, W, bias, residual, Cout, M, N, K);
        }
    }
    switch (epilogue) {            // narrow outputs: single-CTA 128 x 128 tiles
        case 0: return launch_gemm<128, 0, 2, 1>(ctx, A, W, bias, residual, Cout, M, N, K);
        case 1: return launch_gemm<128, 1, 2, 1>(ctx, A, W, bias, residual, Cout, M, N, K);
        default: return launch_gemm<128, 2, 4, 1>(ctx, A, W, bias, residual, Cout, M, N, K);
    }
}

// qkv = A W^T with RoPE applied to the q and k heads in the epilogue (EPI 5); N = 3H, H % 64 == 0, N % 256 == 0 not needed
// (boxes are 64 columns = one head).  table: float2 [32][512] pair-major (cos, sin); pos: int [M].
int gemm_bf16_rope_impl(anon_ctx* ctx, const __nv_bfloat16* A, const __nv_bfloat16* W, const int* pos, const float2* table,
                        void* Cout, int M, int N, int K)
{
    if (!ctx || !A || !W || !pos || !table || !Cout || M < 0 || N <= 128 || K <= 0) return ANON_ERR_INVALID_ARG;
    if (K % BK != 0 || N % 192 != 0) return ANON_ERR_UNSUPPORTED;
    if (M == 0) return ANON_OK;
    LnArgs ln; ln.rope_tab = table; ln.rope_pos = pos;
    return launch_gemm<256, 5, 2, 2>(ctx, A, W, nullptr, nullptr, Cout, M, N, K, &ln);
}

// C = A W^T + bias + LN(res_y; stats, gamma, beta): the residual stream is kept UN-normalised (res_y, with per-row
// (mean, rstd) in res_stats) and normalised on the fly in the epilogue; C may alias res_y.  N > 128 only.
int gemm_bf16_res_ln_impl(anon_ctx* ctx, const __nv_bfloat16* A, const __nv_bfloat16* W, const float* bias, const float* res_y,
                          const float2* res_stats, const float* gamma, const float* beta, float* C, int M, int N, int K)
{
    if (!ctx || !A || !W || !bias || !res_y || !C || M < 0 || N <= 128 || K <= 0 || (res_stats && (!gamma || !beta)))
        return ANON_ERR_INVALID_ARG;
    if (K % BK != 0 || N % 8 != 0 || (res_stats && N > 1024)) return ANON_ERR_UNSUPPORTED;
    if (M == 0) return ANON_OK;
    LnArgs ln; ln.gamma = gamma; ln.beta = beta; ln.res_stats = res_stats;
    if (K >= 2048) return launch_gemm<256, 2, 2, 2>(ctx, A, W, bias, res_y, C, M, N, K, &ln);
    return launch_gemm<256, 2, 5, 2>(ctx, A, W, bias, res_y, C, M, N, K, &ln);      // 5 boxes per warp + 4 mainloop stages
}

// ---- LayerNorm folded into the GEMMs (see the FOLD note above the kernel); H = 768 / 1024 shapes of the encoder ----
// Producer: C = A W^T + bias + LN(res_y) as FP32, Cb = bf16(C), part_out[row][N / 256] = partial (sum, sum of squares).
// The residual's (mean, rstd) come from part_in (partial sums) or res_stats (finished pairs); both NULL: res_y is already normalised.
int gemm_bf16_fold_res_impl(anon_ctx* ctx, const __nv_bfloat16* A, const __nv_bfloat16* W, const float* bias, const float* res_y,
                            const float2* part_in, const float2* res_stats, const float* gamma, const float* beta, float eps, float* C,
                            __nv_bfloat16* Cb, float2* part_out, int M, int N, int K)
{
    if (!ctx || !A || !W || !bias || !res_y || !C || !Cb || !part_out || M < 0 || K <= 0 || ((part_in || res_stats) && (!gamma || !beta)) ||
        (part_in && res_stats))
        return ANON_ERR_INVALID_ARG;
    if (K % BK != 0 || N % 256 != 0 || N > 1024 || N < 256) return ANON_ERR_UNSUPPORTED;
    if (M == 0) return ANON_OK;
    LnArgs ln; ln.gamma = gamma; ln.beta = beta; ln.part_in = part_in; ln.res_stats = res_stats; ln.stat_cnt = N / 256; ln.stat_cols = N; ln.eps = eps;
    ln.part_out = part_out; ln.yb_out = Cb;
    if (K >= 2048) return launch_gemm<256, 2, 2, 2, true>(ctx, A, W, bias, res_y, C, M, N, K, &ln);
    return launch_gemm<256, 2, 4, 2, true>(ctx, A, W, bias, res_y, C, M, N, K, &ln);
}

// Consumer: C = epilogue(LN(A_raw) W^T + b) computed as rstd * (A_raw W'^T - mean * s) + c; W' = bf16(W * gamma), s[n] = sum_k W'[n,k],
// c[n] = b[n] + sum_k beta[k] W[n,k] are prepared at weights load; part_in[row][stat_cols / 256] are the rows' partial statistics.
int gemm_bf16_fold_impl(anon_ctx* ctx, const __nv_bfloat16* A_raw, const __nv_bfloat16* Wf, const float* c, const float* s_vec,
                        const float2* part_in, int stat_cols, float eps, void* C, int M, int N, int K)
{
    if (!ctx || !A_raw || !Wf || !c || !s_vec || !part_in || !C || M < 0 || N <= 128 || K <= 0) return ANON_ERR_INVALID_ARG;
    if (K % BK != 0 || N % 8 != 0 || stat_cols % 256 != 0) return ANON_ERR_UNSUPPORTED;
    if (M == 0) return ANON_OK;
    LnArgs ln; ln.part_in = part_in; ln.stat_cnt = stat_cols / 256; ln.stat_cols = stat_cols; ln.eps = eps; ln.fold_s = s_vec;
    return launch_gemm<256, 0, 2, 2, true>(ctx, A_raw, Wf, c, nullptr, C, M, N, K, &ln);
}

extern "C" int anon_gemm_bf16(anon_ctx* ctx, const void* d_A, const void* d_W, const float* d_bias,
                              const float* d_residual, void* d_C, int32_t M, int32_t N, int32_t K, int32_t epilogue)
{
    if (!ctx) return ANON_ERR_INVALID_ARG;
    CU_TRY(ctx, cudaSetDevice(ctx->device));
    return gemm_bf16_impl(ctx, (const __nv_bfloat16*)d_A, (const __nv_bfloat16*)d_W, d_bias, d_residual, d_C, M, N, K,
                          epilogue);
}

// ---- the fold's two GEMMs exposed for parity tests and per-kernel measurements (include/anonshield.h) ----
extern "C" int anon_gemm_bf16_fold_res(anon_ctx* ctx, const void* d_A, const void* d_W, const float* d_bias, const float* d_res,
                                       const float* d_res_part, const float* d_res_stats, const float* d_gamma, const float* d_beta,
                                       float eps, float* d_C, void* d_Cb, float* d_part_out, int32_t M, int32_t N, int32_t K)
{
    if (!ctx) return ANON_ERR_INVALID_ARG;
    CU_TRY(ctx, cudaSetDevice(ctx->device));
    return gemm_bf16_fold_res_impl(ctx, (const __nv_bfloat16*)d_A, (const __nv_bfloat16*)d_W, d_bias, d_res, (const float2*)d_res_part,
                                   (const float2*)d_res_stats, d_gamma, d_beta, eps, d_C, (__nv_bfloat16*)d_Cb, (float2*)d_part_out, M, N, K);
}

extern "C" int anon_gemm_bf16_fold(anon_ctx* ctx, const void* d_A_raw, const void* d_Wf, const float* d_c, const float* d_s,
                                   const float* d_part, int32_t stat_cols, float eps, void* d_C, int32_t M, int32_t N, int32_t K)
{
    if (!ctx) return ANON_ERR_INVALID_ARG;
    CU_TRY(ctx, cudaSetDevice(ctx->device));
    return gemm_bf16_fold_impl(ctx, (const __nv_bfloat16*)d_A_raw, (const __nv_bfloat16*)d_Wf, d_c, d_s, (const float2*)d_part, stat_cols, eps,
                               d_C, M, N, K);
}
