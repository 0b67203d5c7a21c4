// attention_bf16.cu -- K3: packed variable-length bidirectional self-attention, d_head = 64 (S8a A3; S8c O1).
// No padding FLOPs: the work list holds one item per (sequence, 128-query tile), longest sequences first; keys
// are walked in 64-key chunks up to the sequence's own length only.
//
// sm_100a design (BF16 path): persistent CTAs, two per SM (97 KB shared memory, 256 TMEM columns each), looping
// over (work item, head) units.  Warp-specialised:
//   warp 0      TMA producer : Q tile [128 x 64] (double-buffered) and K / V chunks [64 x 64] of the packed qkv tensor,
//                              128B swizzle, mbarrier completion.  K and V have 3-slot rings of their own and the K
//                              loads run two chunks ahead of the V loads (see the producer)
//   warp 1      MMA issuer   : S = Q K^T   tcgen05.mma M128 N64 K16 x4, both operands K-major in shared memory,
//                                          accumulator = one of two 64-column S buffers in TMEM
//                              O += P V    A = P read from TMEM (BF16 pairs the softmax warps write into P columns of their
//                                          own), B = V chunk, MN-major descriptor
//                              QK^T runs TWO chunks ahead of PV: S(g+2) is issued as soon as the softmax warps have S(g) in
//                              registers, so a finished chunk never waits for the tensor pipe's round trip.  The whole warp
//                              walks the cursors in uniform control flow, the barrier probes of a step are issued together,
//                              and one elected lane issues the MMAs / commits (straight UTCHMMA x4 + UTCBAR in the SASS)
//   warps 2-5   softmax      : one thread per query row: tcgen05.ld S -> exp2 (1/sqrt(64)*log2(e) folded in) -> row sum
//                              -> BF16 P -> tcgen05.st.  A unit's FIRST chunk takes the row maximum of its 64 scores as the
//                              row's reference; every later chunk exponentiates against that reference WITHOUT looking for
//                              its own maximum (33 FMNMX and their chain per chunk), with the second 32 scores loading under
//                              the exponentials of the first 32.  A reference that is too low shows in the chunk's row sum,
//                              which is computed anyway: above 2^18 (also inf / NaN) the scores are read again (S is handed
//                              back only after this decision), the reference is raised to the chunk maximum, O is rescaled
//                              in TMEM (out of line) and the exponentials are repeated.  P, l and O share the reference, so
//                              O / l is exact whatever it is; in between P <= 2^18 per element is far from any FP32 / BF16
//                              range limit.  (The banded kernel keeps the maximum-first order: its rows may not have seen a
//                              key yet.)  The barriers of the NEXT steps (S(g+1) there, PV(g-2) done) are probed right
//                              after the load and looked at only where needed.  O / l of a unit is written after the first
//                              chunk of the next one (the last P V is hidden): BF16 rows into a swizzled 4 KB box per warp,
//                              ONE TMA store of full 128-byte lines (a partly filled last warp stores its rows itself).
//                              The chunk body exists twice (first chunk of a unit / loop over the rest) so that the
//                              write-back and the rare O rescale are not part of the hot loop.
// TMEM per CTA: S 2 x 64 | P 2 x 32 | O 64 = 256 columns.
// Measured with the kernel's own clock64 counters and timing-only ablations (profiles/r02_attention.md, section 5): what bounds
// the kernel is the serial chain of ONE softmax warp per 128 x 64 chunk, ~1,600-1,850 cycles (64 ex2 at 8 issue cycles each on
// the sub-partition's MUFU unit = 512, ~220 other instructions, the rest dependency and barrier latency with only two such warps
// per scheduler); the MMA issuer's own chain is ~1,000 cycles per chunk (1,500 before it was made warp-uniform), the K / V loads
// are not on the path (no change with the loads removed), nor is the tensor pipe (28 %) or TMEM.
#include "common.cuh"
#include "ptx_sm100.cuh"

#include <algorithm>
#include <type_traits>
#include <vector>

namespace {

constexpr int kQT = 128;    // queries per work item
constexpr int kKC = 64;     // keys per chunk
constexpr int kD = 64;
constexpr int kKStages = 3;     // K and V chunks travel in rings of their own: a K slot is free again after QK^T of its chunk,
constexpr int kVStages = 3;     // a V slot after P V -- two chunks later -- so each load is issued three chunk-times before its use
constexpr int kAttThreads = 192;
constexpr int kQBytes = kQT * kD * 2;          // 16 KB
constexpr int kKVBytes = kKC * kD * 2;         // 8 KB (K and V each)
constexpr int kOBytes = kQT * kD * 2;          // 16 KB: the normalised BF16 output tile, staged for the TMA store (one 4 KB box per warp)
constexpr int kAttSmem = 2 * kQBytes + (kKStages + kVStages) * kKVBytes + kOBytes + 1024 /*align slack*/ + 256 /*barriers*/;
// ANON_NVCC_EXTRA=-DATT_PROF=1 builds clock64 counters into the MMA issuer and two softmax warps of virtual CTA 0 (cycles per
// chunk spent in each wait and phase) and exports anon_debug_att_prof; `python kernel_bench.py --only attention --att-prof` prints them
#ifndef ATT_PROF
#define ATT_PROF 0
#endif
#ifndef ATT_ABL
#define ATT_ABL 0               // timing-only ablations (results wrong), never set in the product build: 1 = no ex2, 8 = the
                                // softmax warps only do the barrier handshakes (every warp takes the padding path)
#endif
constexpr int kAttTmemCols = 256;              // S 2 x 64 | P 2 x 32 | O 64

// rows relative to the chunk.  Global attention: kv_row0 = the sequence's first row, n = its length.  Local (band) attention
// (NEXT-3, D20): kv_row0 = first key row any query of the tile may see, n = keys from there, and q_valid carries
// (q_row0 - kv_row0) << 8 in its upper bits: query row r sees key kk (relative to kv_row0) iff |kk - (delta + r)| <= band.
#if ATT_PROF
__device__ unsigned long long g_att_prof[64];
#define PROF_T(v) const long long v = clock64()
#define PROF_ADD(i, a, b) do { if (blockIdx.x == 0) prof[i] += (unsigned long long)((b) - (a)); } while (0)
#else
#define PROF_T(v)
#define PROF_ADD(i, a, b)
#endif
struct WorkItem { int q_row0; int kv_row0; int n; int q_valid; };
constexpr int kBand = 64;   // half width of the local window the tcgen05 kernel supports (window 128)

__device__ __forceinline__ float ex2f(float x) { float y; asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float max3(float a, float b, float c) {
    float d; asm("max.f32 %0, %1, %2, %3;" : "=f"(d) : "f"(a), "f"(b), "f"(c)); return d;
}
__device__ __forceinline__ uint64_t pk2(float a, float b) { uint64_t r; asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(a), "f"(b)); return r; }
__device__ __forceinline__ void upk2(uint64_t v, float& a, float& b) { asm("mov.b64 {%0, %1}, %2;" : "=f"(a), "=f"(b) : "l"(v)); }
__device__ __forceinline__ uint64_t fma2(uint64_t a, uint64_t b, uint64_t c) {
    uint64_t d; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c)); return d;
}
__device__ __forceinline__ uint64_t add2(uint64_t a, uint64_t b) {
    uint64_t d; asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b)); return d;
}
__device__ __forceinline__ uint32_t pack2(float a, float b) {
    __nv_bfloat162 v = __floats2bfloat162_rn(a, b);
    return *reinterpret_cast<uint32_t*>(&v);
}

// O *= alpha for this thread's row (64 FP32 columns in TMEM).  Rare (the reference maximum moved by more than 2^8 after a unit's
// first chunk) and deliberately NOT inlined: its 32 extra live registers would otherwise be part of the hot loop's allocation.
__device__ __noinline__ void rescale_o(uint32_t taddr, float alpha) {
#pragma unroll
    for (int hh = 0; hh < 2; hh++) {
        uint32_t o[32];
        ptx::tmem_ld_32x32b_x32(taddr + 32u * hh, o);
        ptx::tmem_ld_wait();
#pragma unroll
        for (int j = 0; j < 32; j++) o[j] = __float_as_uint(__uint_as_float(o[j]) * alpha);
        ptx::tmem_st_32x32b_x32(taddr + 32u * hh, o);
    }
    ptx::tmem_st_wait();
}

template <bool BAND>
__global__ void __launch_bounds__(kAttThreads, 2)
attention_tcgen05_kernel(const __grid_constant__ CUtensorMap tmap_q, const __grid_constant__ CUtensorMap tmap_kv,
                         const __grid_constant__ CUtensorMap tmap_o, const WorkItem* __restrict__ work, int n_units, int heads, int H, __nv_bfloat16* __restrict__ ctx)
{
    extern __shared__ uint8_t smem_raw[];
    const uint32_t smem_base = (ptx::smem_u32(smem_raw) + 1023u) & ~1023u;
    const uint32_t q_smem = smem_base;                                   // 2 x 16 KB
    const uint32_t k_smem = smem_base + 2 * kQBytes;                     // K ring: stages x 8 KB
    const uint32_t v_smem = k_smem + kKStages * kKVBytes;                // V ring: stages x 8 KB
    const uint32_t o_smem = v_smem + kVStages * kKVBytes;                // 4 x 4 KB: [32 rows x 128 B], 128B swizzle, one box per softmax warp
    const uint32_t bar_base = o_smem + kOBytes;
    auto q_full = [&](uint32_t i) { return bar_base + 8u * i; };
    auto q_empty = [&](uint32_t i) { return bar_base + 8u * (2 + i); };
    auto k_full = [&](uint32_t i) { return bar_base + 8u * (4 + i); };
    auto v_full = [&](uint32_t i) { return bar_base + 8u * (24 + i); };
    auto k_empty = [&](uint32_t i) { return bar_base + 8u * (8 + i); };     // QK^T of the chunk in K slot i has completed
    auto v_empty = [&](uint32_t i) { return bar_base + 8u * (28 + i); };    // P V of the chunk in V slot i has completed
    auto s_full = [&](uint32_t i) { return bar_base + 8u * (12 + i); };    // S chunk computed (MMA commit)
    auto p_full = [&](uint32_t i) { return bar_base + 8u * (14 + i); };    // P chunk written (4 softmax warps)
    auto pv_done = [&](uint32_t i) { return bar_base + 8u * (16 + i); };   // PV of the chunk in P buffer i has completed
    auto s_free = [&](uint32_t i) { return bar_base + 8u * (22 + i); };    // S buffer i has been read into registers (4 warps)
    const uint32_t o_full = bar_base + 8u * 18, o_empty = bar_base + 8u * 20;
    const uint32_t tmem_slot = bar_base + 8u * 19;
    uint32_t* tmem_slot_ptr = reinterpret_cast<uint32_t*>(smem_raw + (tmem_slot - ptx::smem_u32(smem_raw)));

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    // unit u = item * heads + head.  The roles step u by gridDim.x; (item, head) follow by addition (two integer divisions per
    // thread here instead of one or two per unit -- ~40 instructions each -- in every role)
    const int step_item = (int)gridDim.x / heads, step_head = (int)gridDim.x % heads;
    const int item0 = (int)blockIdx.x / heads, head0 = (int)blockIdx.x % heads;
    auto next_unit = [&](int& item, int& head) { item += step_item; head += step_head; if (head >= heads) { head -= heads; item++; } };

    if (warp == 0 && lane == 0) {
        ptx::prefetch_tensormap(&tmap_q);
        ptx::prefetch_tensormap(&tmap_kv);
        ptx::prefetch_tensormap(&tmap_o);
    }
    if (warp == 1 && lane == 0) {
        for (uint32_t i = 0; i < 2; i++) {
            ptx::mbar_init(q_full(i), 1); ptx::mbar_init(q_empty(i), 1);
            ptx::mbar_init(s_full(i), 1); ptx::mbar_init(p_full(i), 4); ptx::mbar_init(pv_done(i), 1);
            ptx::mbar_init(s_free(i), 4);
        }
        ptx::mbar_init(o_full, 1); ptx::mbar_init(o_empty, 4);
        for (uint32_t i = 0; i < kKStages; i++) { ptx::mbar_init(k_full(i), 1); ptx::mbar_init(k_empty(i), 1); }
        for (uint32_t i = 0; i < kVStages; i++) { ptx::mbar_init(v_full(i), 1); ptx::mbar_init(v_empty(i), 1); }
        ptx::fence_barrier_init();
        ptx::fence_proxy_async();
    }
    if (warp == 2) {
        ptx::tmem_alloc(tmem_slot, kAttTmemCols);
        ptx::tmem_relinquish();
    }
    ptx::tc_fence_before();
    __syncthreads();
    ptx::tc_fence_after();
    // TMEM columns: S buffers 2 x 64 (FP32 scores) | P buffers 2 x 32 (BF16 pairs, 64 keys each) | O 64 (FP32 accumulator)
    const uint32_t tmem_base = *tmem_slot_ptr;
    const uint32_t tmem_p = tmem_base + 128u;
    const uint32_t tmem_o = tmem_base + 192u;

    if (warp == 0) {
        // ===== TMA producer: two cursors over the flattened (unit, chunk) sequence.  The K cursor runs two chunks ahead of the
        // V cursor -- the distance between QK^T and P V in the MMA issuer -- so that neither ring waits on the other's slot: a K
        // (V) slot is re-filled as soon as the QK^T (P V) that read it has completed, four chunk-times before its next use.  With K
        // and V in one slot the re-fill could only start after P V, ONE chunk-time before the next QK^T needed it, and the kernel
        // ran at the TMA round trip per chunk (profiles/r02_attention.md, section 5) =====
        if (lane == 0) {
            struct Cur { int u, item, head, c, nc; uint32_t qi, g; WorkItem w; };
            auto enter = [&](Cur& k) { if (k.u < n_units) { k.w = work[k.item]; k.nc = (k.w.n + kKC - 1) / kKC; } };
            auto advance = [&](Cur& k) {
                k.g++;
                if (++k.c == k.nc) { k.u += gridDim.x; next_unit(k.item, k.head); k.qi++; k.c = 0; enter(k); }
            };
            Cur a{(int)blockIdx.x, item0, head0, 0, 0, 0u, 0u, WorkItem{0, 0, 0, 0}};
            enter(a);
            Cur b = a;
            auto load_k = [&]() {
                const int head = a.head;
                if (a.c == 0) {
                    const uint32_t qb = a.qi & 1u;
                    ptx::mbar_wait_backoff(q_empty(qb), ((a.qi >> 1) & 1u) ^ 1u);
                    ptx::mbar_arrive_expect_tx(q_full(qb), kQBytes);
                    ptx::tma_load_2d(q_smem + qb * kQBytes, &tmap_q, q_full(qb), head * kD, a.w.q_row0);
                }
                const uint32_t st = a.g % kKStages;
                ptx::mbar_wait_backoff(k_empty(st), ((a.g / kKStages) & 1u) ^ 1u);
                ptx::mbar_arrive_expect_tx(k_full(st), kKVBytes);
                ptx::tma_load_2d(k_smem + st * kKVBytes, &tmap_kv, k_full(st), H + head * kD, a.w.kv_row0 + a.c * kKC);
                advance(a);
            };
            auto load_v = [&]() {
                const int head = b.head;
                const uint32_t st = b.g % kVStages;
                ptx::mbar_wait_backoff(v_empty(st), ((b.g / kVStages) & 1u) ^ 1u);
                ptx::mbar_arrive_expect_tx(v_full(st), kKVBytes);
                ptx::tma_load_2d(v_smem + st * kKVBytes, &tmap_kv, v_full(st), 2 * H + head * kD, b.w.kv_row0 + b.c * kKC);
                advance(b);
            };
            if (a.u < n_units) load_k();
            if (a.u < n_units) load_k();
            while (b.u < n_units) {
                if (a.u < n_units) load_k();
                load_v();
            }
        }
    } else if (warp == 1) {
        // ===== MMA issuer: two cursors over the flattened (unit, chunk) sequence.  QK^T runs TWO chunks ahead of PV: S(g+2) is
        // issued as soon as the softmax warps have pulled S(g) into registers (s_free), not when P(g) has been consumed -- P has
        // TMEM columns of its own -- so a finished chunk never waits for the tensor pipe's round trip.
        // The WHOLE warp walks the cursors in uniform control flow and one elected lane issues: with the loop inside
        // `if (lane == 0)` ptxas cannot prove the descriptors warp-uniform and wraps every tcgen05.mma / commit in an
        // ELECT ... BRA.U.ANY loop -- measured with clock64 at 485 + 440 cycles per chunk for 8 MMAs and 5 commits, which made this
        // thread, not the softmax, the pace of the kernel (profiles/r02_attention.md, section 5) =====
        {
            constexpr uint32_t idesc_qk = ptx::make_idesc_bf16(kQT, kKC);          // both operands K-major
            constexpr uint32_t idesc_pv = ptx::make_idesc_bf16(kQT, kD, 1);        // B = V is MN-major
            // nc_next = chunk count of the unit after the cursor's, loaded one unit ahead so that no MMA waits on it
            // (item, head) = the unit AFTER the cursor's: where nc_next comes from
            struct Cur { int u, item, head, c, nc, nc_next; uint32_t qi, g; };
            // (the shuffle -- at the point of use, a whole unit after the load -- tells ptxas the count is warp-uniform)
            auto chunks_of = [&](int u, int item) { return u < n_units ? (work[item].n + kKC - 1) / kKC : 0; };
            auto advance = [&](Cur& k) {
                k.g++;
                if (++k.c == k.nc) {
                    k.u += gridDim.x; k.qi++; k.c = 0;
                    k.nc = __shfl_sync(0xffffffffu, k.nc_next, 0);
                    next_unit(k.item, k.head);
                    k.nc_next = chunks_of(k.u + (int)gridDim.x, k.item);
                }
            };
            Cur a{(int)blockIdx.x, item0, head0, 0, __shfl_sync(0xffffffffu, chunks_of((int)blockIdx.x, item0), 0), 0, 0u, 0u};
            next_unit(a.item, a.head);
            a.nc_next = chunks_of(a.u + (int)gridDim.x, a.item);
            Cur b = a;
#if ATT_PROF
            unsigned long long prof[16];
            for (int i = 0; i < 16; i++) prof[i] = 0;
            const long long t_begin = clock64();
#endif
            auto issue_qk = [&]() {
                const uint32_t qb = a.qi & 1u, st = a.g % kKStages, sb = a.g & 1u;
                PROF_T(t0);
                // the probes are issued together (an mbarrier probe answers after ~70 cycles even when the phase is long complete)
                // and only a failed one is waited for
                const bool ok_s = a.g < 2u || ptx::mbar_try_wait(s_free(sb), ((a.g - 2u) >> 1) & 1u);   // S(g-2) has left this buffer
                const bool ok_k = ptx::mbar_try_wait(k_full(st), (a.g / kKStages) & 1u);
                const bool ok_q = a.c != 0 || ptx::mbar_try_wait(q_full(qb), (a.qi >> 1) & 1u);
                PROF_T(t1);
                if (!ok_s) ptx::mbar_wait(s_free(sb), ((a.g - 2u) >> 1) & 1u);
                if (!ok_q) ptx::mbar_wait(q_full(qb), (a.qi >> 1) & 1u);
                PROF_T(t2);
                if (!ok_k) ptx::mbar_wait(k_full(st), (a.g / kKStages) & 1u);
                PROF_T(t3);
                PROF_ADD(0, t0, t1); PROF_ADD(1, t1, t2); PROF_ADD(2, t2, t3);
                ptx::tc_fence_after();
                const uint64_t qd = ptx::make_desc_k_sw128(q_smem + qb * kQBytes);
                const uint64_t kd = ptx::make_desc_k_sw128(k_smem + st * kKVBytes);
                if (ptx::elect_one()) {
#pragma unroll
                    for (int k = 0; k < kD / 16; k++)
                        ptx::mma_f16_ss(tmem_base + sb * 64u, qd + (uint64_t)(2 * k), kd + (uint64_t)(2 * k), idesc_qk, k ? 1u : 0u);
                    PROF_T(tm);
                    PROF_ADD(10, t3, tm);
                    ptx::mma_commit(s_full(sb));
                    ptx::mma_commit(k_empty(st));
                    if (a.c == a.nc - 1) ptx::mma_commit(q_empty(qb));   // last use of this Q tile
                }
                __syncwarp();
                PROF_T(t4);
                PROF_ADD(3, t3, t4);
            };
            auto issue_pv = [&]() {
                const uint32_t st = b.g % kVStages, sb = b.g & 1u;
                PROF_T(t0);
                const bool ok_v = ptx::mbar_try_wait(v_full(st), (b.g / kVStages) & 1u);
                const bool ok_p = ptx::mbar_try_wait(p_full(sb), (b.g >> 1) & 1u);
                const bool ok_o = b.c != 0 || ptx::mbar_try_wait(o_empty, (b.qi & 1u) ^ 1u);   // the previous unit's O has been read (finalize)
                PROF_T(t1);
                if (!ok_v) ptx::mbar_wait(v_full(st), (b.g / kVStages) & 1u);
                if (!ok_p) ptx::mbar_wait(p_full(sb), (b.g >> 1) & 1u);
                PROF_T(t2);
                if (!ok_o) ptx::mbar_wait(o_empty, (b.qi & 1u) ^ 1u);
                PROF_T(t3);
                PROF_ADD(4, t0, t1); PROF_ADD(5, t1, t2); PROF_ADD(6, t2, t3);
                ptx::tc_fence_after();
                const uint64_t vd = ptx::make_desc_mn_sw128(v_smem + st * kKVBytes);
                if (ptx::elect_one()) {
#pragma unroll
                    for (int k = 0; k < kKC / 16; k++)                   // 16 keys per MMA: 8 TMEM columns of P, 2 KB of V
                        ptx::mma_f16_ts(tmem_o, tmem_p + sb * 32u + 8u * k, vd + (uint64_t)(128 * k), idesc_pv, (b.c | k) ? 1u : 0u);
                    PROF_T(tm);
                    PROF_ADD(11, t3, tm);
                    ptx::mma_commit(v_empty(st));
                    ptx::mma_commit(pv_done(sb));
                    if (b.c == b.nc - 1) ptx::mma_commit(o_full);
                }
                __syncwarp();
                PROF_T(t4);
                PROF_ADD(7, t3, t4);
                PROF_ADD(9, 0, 1);
            };
            if (a.nc) { issue_qk(); advance(a); }
            if (a.nc) { issue_qk(); advance(a); }
            while (b.nc) {
                if (a.nc) { issue_qk(); advance(a); }        // S(g+2): gated by s_free(g), early in the softmax of chunk g
                issue_pv();                                  // PV(g): gated by p_full(g), the end of that softmax
                PROF_T(ta);
                advance(b);
                PROF_T(tb);
                PROF_ADD(12, ta, tb);
            }
#if ATT_PROF
            if (blockIdx.x == 0 && lane == 0) { prof[8] = (unsigned long long)(clock64() - t_begin); for (int i = 0; i < 16; i++) g_att_prof[i] = prof[i]; }
#endif
        }
    } else {
        // ===== softmax warps: thread = query row =====
        const uint32_t quarter = (uint32_t)(warp & 3);
        const uint32_t lane_base = (quarter * 32u) << 16;
        const int row = (int)quarter * 32 + lane;
        const float sc = 0.125f * 1.4426950408889634f;                   // 1/sqrt(64) * log2(e)
        uint32_t qi = 0, g = 0;
        bool s_ok = false;                                               // s_full of the chunk about to start has been seen (probed early)
        bool pend = false;
        uint32_t pend_par = 0;
        float pend_l = 1.f;
        int pend_row0 = 0, pend_valid = 0, pend_head = 0;
        auto finalize = [&]() {                                          // O / l -> BF16 row of ctx
            ptx::mbar_wait(o_full, pend_par);
            ptx::tc_fence_after();
            uint32_t o[64];
            ptx::tmem_ld_32x32b_x32(tmem_o + lane_base, o);
            ptx::tmem_ld_32x32b_x32(tmem_o + lane_base + 32u, o + 32);
            ptx::tmem_ld_wait();
            ptx::tc_fence_before();
            __syncwarp();
            if (lane == 0) ptx::mbar_arrive(o_empty);
            float inv;                                                   // the row sum is >= 1 (the reference key's own 2^0 at least)
            asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(inv) : "f"(pend_l));
            if ((int)quarter * 32 + 32 <= pend_valid) {
                // all 32 rows of this warp are real: BF16 rows into the warp's swizzled 4 KB box, ONE TMA store of full 128-byte lines.
                // (Per-thread 16-byte stores put 32 different lines into every store instruction: with them the write-back cost
                // 10 % of the kernel at n = 512 and 17 % of the banded one, profiles/r02_attention.md section 5.)
                if (lane == 0) ptx::bulk_wait_read<0>();                 // the box's previous store has read it (a unit ago)
                __syncwarp();
                const uint32_t box = o_smem + quarter * 4096u, rowb = box + (uint32_t)lane * 128u, sw = (uint32_t)(lane & 7);
#pragma unroll
                for (int v = 0; v < 8; v++)
                    asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(rowb + ((((uint32_t)v) ^ sw) << 4)),
                                 "r"(pack2(__uint_as_float(o[8 * v]) * inv, __uint_as_float(o[8 * v + 1]) * inv)),
                                 "r"(pack2(__uint_as_float(o[8 * v + 2]) * inv, __uint_as_float(o[8 * v + 3]) * inv)),
                                 "r"(pack2(__uint_as_float(o[8 * v + 4]) * inv, __uint_as_float(o[8 * v + 5]) * inv)),
                                 "r"(pack2(__uint_as_float(o[8 * v + 6]) * inv, __uint_as_float(o[8 * v + 7]) * inv)) : "memory");
                ptx::fence_proxy_async();
                __syncwarp();
                if (lane == 0) {
                    ptx::tma_store_2d(&tmap_o, box, pend_head * kD, pend_row0 + (int)quarter * 32);
                    ptx::bulk_commit();
                }
            } else if (row < pend_valid) {                               // the tile's last, partly filled warp: its rows one by one
                uint4* dst = reinterpret_cast<uint4*>(ctx + (size_t)(pend_row0 + row) * H + pend_head * kD);
#pragma unroll
                for (int v = 0; v < 8; v++)
                    dst[v] = make_uint4(pack2(__uint_as_float(o[8 * v]) * inv, __uint_as_float(o[8 * v + 1]) * inv),
                                        pack2(__uint_as_float(o[8 * v + 2]) * inv, __uint_as_float(o[8 * v + 3]) * inv),
                                        pack2(__uint_as_float(o[8 * v + 4]) * inv, __uint_as_float(o[8 * v + 5]) * inv),
                                        pack2(__uint_as_float(o[8 * v + 6]) * inv, __uint_as_float(o[8 * v + 7]) * inv));
            }
            pend = false;
        };
#if ATT_PROF
        unsigned long long prof[16];
        for (int i = 0; i < 16; i++) prof[i] = 0;
        const long long t_begin = clock64();
#endif
        WorkItem wn = work[min((int)blockIdx.x, n_units - 1) / heads];         // next unit's item, loaded one unit ahead
        int item_n = item0, head_n = head0;                              // (item, head) of the unit after this one
        for (int u = blockIdx.x; u < n_units; u += gridDim.x, qi++) {
            const WorkItem w = wn;
            const int head = head_n;
            next_unit(item_n, head_n);
            if (u + (int)gridDim.x < n_units) wn = work[item_n];
            const int nc = (w.n + kKC - 1) / kKC;
            float m = -INFINITY, l = 0.f;                                // reference max (scaled, log2 domain), row sum
            // One chunk.  The body is instantiated twice -- for a unit's first chunk, after which the previous unit's write-back
            // runs, and inside the loop over the others -- so that the write-back (64 more live registers) is not part of the
            // hot loop: with it inlined there the whole loop was allocated and scheduled around it (n = 512: 0.665 -> 0.60 ms
            // with the write-back's arithmetic removed, far more than that arithmetic takes)
            auto chunk = [&](auto first_tag, const int c) {
                constexpr bool FIRST = decltype(first_tag)::value;
                // SPEC: after a unit's first chunk the exponentials are taken against the reference the row already has, WITHOUT
                // looking for the chunk's maximum first (33 FMNMX and their dependency chain per chunk); a reference that is too
                // low for this chunk shows in the chunk's row sum, which is computed anyway, and only then -- rare -- the scores
                // are read again, the reference is raised (O rescaled) and the exponentials repeated.  The S buffer is therefore
                // handed back (s_free) only after that decision.  Not in the banded kernel (rows that have not seen a key yet).
                constexpr bool SPEC = !FIRST && !BAND;
                const uint32_t sb = g & 1u;
                const uint32_t t_s = tmem_base + lane_base + sb * 64u;
                PROF_T(t0);
                if (!s_ok) ptx::mbar_wait(s_full(sb), (g >> 1) & 1u);
                s_ok = false;
                PROF_T(t1);
                PROF_ADD(0, t0, t1);
                ptx::tc_fence_after();
                if (ATT_ABL == 8 || (int)quarter * 32 >= (w.q_valid & 0xff)) {           // no query of this warp is real: P rows are don't-care
                    ptx::tc_fence_before();
                    __syncwarp();
                    if (lane == 0) ptx::mbar_arrive(s_free(sb));
                    // like the working warps, do not signal P(g) before PV(g-2) is done: a warp that ran two chunks ahead
                    // would otherwise arrive on the phase of chunk g-2 and let PV start before the others have written P
                    if (g >= 2u) ptx::mbar_wait(pv_done(sb), ((g - 2u) >> 1) & 1u);
                    __syncwarp();
                    if (lane == 0) ptx::mbar_arrive(p_full(sb));
                    return;
                }
                uint32_t r[64];
                const int valid = w.n - c * kKC;                         // keys of this chunk that belong to the sequence
                auto load_scores = [&]() {
                    ptx::tmem_ld_32x32b_x32(t_s, r);
                    ptx::tmem_ld_32x32b_x32(t_s + 32u, r + 32);          // both loads, ONE wait: taking the maxima of the first 32 scores
                    ptx::tmem_ld_wait();                                 // under the second load costs a second wait and measured slower
                    if (valid < kKC) {
#pragma unroll
                        for (int j = 0; j < kKC; j++) if (j >= valid) r[j] = 0xff800000u;      // -inf
                    }
                    if (BAND) {                                          // keys outside |key - query| <= kBand: -inf
                        const int qq = (w.q_valid >> 8) + row - c * kKC; // the query's own column in this chunk
                        const int jlo = qq - kBand, jhi = qq + kBand;
                        if (jlo > 0 || jhi < kKC - 1) {
#pragma unroll
                            for (int j = 0; j < kKC; j++) if (j < jlo || j > jhi) r[j] = 0xff800000u;
                        }
                    }
                };
                auto release_s = [&]() {                                 // the scores are in registers: S(g+2) may overwrite the buffer
                    ptx::tc_fence_before();
                    __syncwarp();
                    if (lane == 0) ptx::mbar_arrive(s_free(sb));
                };
                // SPEC on a full chunk: the second 32 scores are loaded under the exponentials of the first 32
                const bool piped = SPEC && valid >= kKC;
                if (piped) {
                    ptx::tmem_ld_32x32b_x32(t_s, r);
                    ptx::tmem_ld_wait();
                    ptx::tmem_ld_32x32b_x32(t_s + 32u, r + 32);
                } else {
                    load_scores();
                }
                if (!SPEC) release_s();
                // PV(g-2) has all but always finished by now, and so has QK^T(g+1) (issued one chunk-time ago): probe both barriers
                // here and look at the answers only before the P store / at the top of the next chunk, so that the ~70-150 cycles a
                // probe takes are covered by the maximum and the exponentials (n = 512: 0.656 ms with the early probes, 0.667 without)
                const bool pv_ok = g < 2u || ptx::mbar_test_wait(pv_done(sb), ((g - 2u) >> 1) & 1u);
                s_ok = ptx::mbar_test_wait(s_full(sb ^ 1u), ((g + 1u) >> 1) & 1u);
                PROF_T(t2);
                PROF_ADD(1, t1, t2);
                // the chunk's maximum; raise the reference when it is more than 2^thr above it (first chunk: m = -inf)
                auto raise = [&](const float thr) {
                    float cmx[4];                                        // four independent chains, then a tree
#pragma unroll
                    for (int q4 = 0; q4 < 4; q4++) {
                        cmx[q4] = max3(__uint_as_float(r[16 * q4]), __uint_as_float(r[16 * q4 + 1]), __uint_as_float(r[16 * q4 + 2]));
#pragma unroll
                        for (int j = 3; j + 1 < 16; j += 2)
                            cmx[q4] = max3(cmx[q4], __uint_as_float(r[16 * q4 + j]), __uint_as_float(r[16 * q4 + j + 1]));
                        cmx[q4] = fmaxf(cmx[q4], __uint_as_float(r[16 * q4 + 15]));
                    }
                    const float cm = fmaxf(max3(cmx[0], cmx[1], cmx[2]), cmx[3]);
                    const float mnew = cm * sc;
                    if (__any_sync(0xffffffffu, mnew > m + thr)) {
                        float alpha = 1.0f;
                        if (mnew > m) { alpha = ex2f(m - mnew); m = mnew; l *= alpha; }
                        if (!FIRST) {                                    // rescale O in TMEM once PV(g-1) has landed
                            ptx::mbar_wait(pv_done((g - 1u) & 1u), ((g - 1u) >> 1) & 1u);
                            ptx::tc_fence_after();
                            rescale_o(tmem_o + lane_base, alpha);
                        }
                    }
                };
                uint32_t pk[32];
                auto exps = [&](const bool second_half_in_flight) -> float {     // P = 2^(s * sc - m) as BF16 pairs; returns the row's sum over the chunk
                    uint64_t sum_a = pk2(0.f, 0.f), sum_b = sum_a;       // packed FP32x2 partial row sums
                    // BAND: a row may not have seen any key yet (m = -inf): exponentiate against 0, every p is then 0
                    const float mref = (BAND && m == -INFINITY) ? 0.f : m;
                    const uint64_t sc2 = pk2(sc, sc), nm2 = pk2(-mref, -mref);
#pragma unroll
                    for (int hh = 0; hh < 2; hh++) {
                        if (hh == 1 && second_half_in_flight) ptx::tmem_ld_wait();
                        if (hh == 1 && valid <= 32) {                    // second half of a short last chunk: all masked
#pragma unroll
                            for (int j = 16; j < 32; j++) pk[j] = 0u;
                            break;
                        }
                        if (BAND) {                                      // a half-chunk none of this warp's 32 rows can see
                            const int wq = (w.q_valid >> 8) + (int)quarter * 32 - c * kKC;    // column of the warp's first row
                            if (32 * hh + 31 < wq - kBand || 32 * hh > wq + 31 + kBand) {
#pragma unroll
                                for (int j = 16 * hh; j < 16 * hh + 16; j++) pk[j] = 0u;
                                continue;
                            }
                        }
#pragma unroll
                        for (int j = 16 * hh; j < 16 * hh + 16; j++) {
                            const uint64_t t = fma2(pk2(__uint_as_float(r[2 * j]), __uint_as_float(r[2 * j + 1])), sc2, nm2);
                            float p0, p1;
#if ATT_ABL == 1
                            upk2(t, p0, p1);
#else
                            { float t0, t1; upk2(t, t0, t1); p0 = ex2f(t0); p1 = ex2f(t1); }
#endif
                            if (j & 1) sum_b = add2(sum_b, pk2(p0, p1)); else sum_a = add2(sum_a, pk2(p0, p1));
                            pk[j] = pack2(p0, p1);
                        }
                    }
                    float s0, s1;
                    upk2(add2(sum_a, sum_b), s0, s1);
                    return s0 + s1;
                };
                if (!SPEC) {
                    raise(8.0f);
                    PROF_T(t3);
                    PROF_ADD(2, t2, t3);
                    l += exps(false);
                    PROF_T(t4);
                    PROF_ADD(3, t3, t4);
                } else {
                    float sum = exps(piped);
                    // a P above 2^12 means the reference is more than 12 binades too low for this chunk (also catches inf / NaN)
                    if (__any_sync(0xffffffffu, !(sum <= 4096.0f * (float)kKC))) {
                        load_scores();                                   // S(g) is still there: s_free has not been signalled
                        raise(0.0f);
                        sum = exps(false);
                    }
                    l += sum;
                    release_s();
                    PROF_T(t4);
                    PROF_ADD(3, t2, t4);
                }
                PROF_T(t4b);
                if (!pv_ok) ptx::mbar_wait(pv_done(sb), ((g - 2u) >> 1) & 1u);      // PV(g-2) has finished reading this P buffer
                ptx::tc_fence_after();
                PROF_T(t5);
                PROF_ADD(4, t4b, t5);
                ptx::tmem_st_32x32b_x32(tmem_p + lane_base + sb * 32u, pk);
                ptx::tmem_st_wait();
                ptx::tc_fence_before();
                __syncwarp();
                if (lane == 0) ptx::mbar_arrive(p_full(sb));
                PROF_T(t6);
                PROF_ADD(5, t5, t6);
                PROF_ADD(9, 0, 1);
            };
            chunk(std::true_type{}, 0);
            g++;
            {
                PROF_T(t6);
                if (pend) finalize();
                PROF_T(t7);
                PROF_ADD(6, t6, t7);
            }
#pragma unroll 1
            for (int c = 1; c < nc; c++, g++) chunk(std::false_type{}, c);
            // the O / l write-back of this unit is deferred until after the first chunk of the next one, so that the
            // wait for the last PV overlaps useful work
            pend = true; pend_par = qi & 1u; pend_l = l;
            pend_row0 = w.q_row0; pend_valid = w.q_valid & 0xff; pend_head = head;
        }
        if (pend) finalize();
        if (lane == 0) ptx::bulk_wait<0>();                              // the last TMA stores have left shared memory and are complete
#if ATT_PROF
        if (blockIdx.x == 0 && warp == 2 && lane == 0) { prof[8] = (unsigned long long)(clock64() - t_begin); for (int i = 0; i < 16; i++) g_att_prof[16 + i] = prof[i]; }
        if (blockIdx.x == 0 && warp == 5 && lane == 31) { prof[8] = (unsigned long long)(clock64() - t_begin); for (int i = 0; i < 16; i++) g_att_prof[32 + i] = prof[i]; }
#endif
    }

    ptx::tc_fence_before();
    __syncthreads();
    if (warp == 2) {
        ptx::tc_fence_after();
        ptx::tmem_dealloc(tmem_base, kAttTmemCols);
    }
}

}  // namespace

// enc::attention_f32_kernel lives in encoder_kernels.cuh (FP32 path); declared here for the dtype-0 branch
#include "encoder_kernels.cuh"

int attention_plan(anon_ctx* ctx, WsCursor& ws, const int32_t* h_cu, int B, int dtype, AttnPlan* plan, int window)
{
    plan->window = window;
    if (window != 0 && dtype == 1 && window != 2 * kBand) return ANON_ERR_UNSUPPORTED;
    // h_cu points at this chunk's first sequence boundary; rows are relative to token h_cu[0]
    plan->d_work = nullptr; plan->n_items = 0; plan->n_rows = 0;
    if (!ctx || !h_cu || B < 0) return ANON_ERR_INVALID_ARG;
    for (int s = 0; s < B; s++)
        if (h_cu[s + 1] < h_cu[s] || h_cu[s + 1] - h_cu[s] > 512) return ANON_ERR_UNSUPPORTED;
    if (dtype == 0 || B == 0) return ANON_OK;
    const int tok0 = h_cu[0];
    plan->n_rows = h_cu[B] - tok0;
    std::vector<WorkItem> items;
    items.reserve((size_t)(h_cu[B] - tok0) / kQT + B);
    for (int s = 0; s < B; s++) {
        const int a = h_cu[s] - tok0, n = h_cu[s + 1] - h_cu[s];
        for (int q0 = 0; q0 < n; q0 += kQT) {
            if (window == 0) { items.push_back(WorkItem{a + q0, a, n, std::min(kQT, n - q0)}); continue; }
            const int k0 = std::max(0, q0 - kBand), k1 = std::min(n, q0 + kQT + kBand);
            items.push_back(WorkItem{a + q0, a + k0, k1 - k0, std::min(kQT, n - q0) | ((q0 - k0) << 8)});
        }
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
        enc::attention_f32_kernel<<<dim3(B, heads, (512 + enc::kF32QueryBlock - 1) / enc::kF32QueryBlock), 128, 0, ctx->stream>>>((const float*)d_qkv, d_cu, 0, tok0, hidden, (float*)d_ctx,
                                                                           plan.window ? plan.window / 2 : -1);
        CU_LAUNCH_CHECK(ctx, "attention_f32_kernel");
        return ANON_OK;
    }
    if (plan.n_items == 0) return ANON_OK;
    // rows of the packed qkv tensor this launch may touch: up to the end of the chunk (plan.n_rows)
    CUtensorMap tq, tkv;
    int rc = make_tmap_2d(ctx, &tq, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, d_qkv, (uint64_t)plan.n_rows, (uint64_t)3 * hidden, kD, kQT);
    if (rc) return rc;
    rc = make_tmap_2d(ctx, &tkv, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, d_qkv, (uint64_t)plan.n_rows, (uint64_t)3 * hidden, kD, kKC);
    if (rc) return rc;
    CUtensorMap to;          // ctx rows for the write-back: boxes of 32 rows x one head (64 columns)
    rc = make_tmap_2d(ctx, &to, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, d_ctx, (uint64_t)plan.n_rows, (uint64_t)hidden, kD, 32);
    if (rc) return rc;
    rc = ensure_smem_attr(ctx, (const void*)attention_tcgen05_kernel<false>, kAttSmem);
    if (rc) return rc;
    rc = ensure_smem_attr(ctx, (const void*)attention_tcgen05_kernel<true>, kAttSmem);
    if (rc) return rc;
    const long long units = (long long)plan.n_items * heads;
    const int grid = (int)std::min<long long>(units, 2LL * ctx->sm_count);
    if (plan.window)
        attention_tcgen05_kernel<true><<<grid, kAttThreads, kAttSmem, ctx->stream>>>(tq, tkv, to, (const WorkItem*)plan.d_work, (int)units,
                                                                                      heads, hidden, (__nv_bfloat16*)d_ctx);
    else
        attention_tcgen05_kernel<false><<<grid, kAttThreads, kAttSmem, ctx->stream>>>(tq, tkv, to, (const WorkItem*)plan.d_work, (int)units,
                                                                                       heads, hidden, (__nv_bfloat16*)d_ctx);
    CU_LAUNCH_CHECK(ctx, "attention_tcgen05_kernel");
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

extern "C" int anon_attention_local(anon_ctx* ctx, const void* d_qkv, const int32_t* d_cu_seqlens, const int32_t* h_cu_seqlens,
                                    int32_t B, int32_t T, int32_t hidden, int32_t heads, int32_t dtype, int32_t window, void* d_ctx)
{
    if (!ctx) return ANON_ERR_INVALID_ARG;
    CU_TRY(ctx, cudaSetDevice(ctx->device));
    if (!h_cu_seqlens || B < 0 || T < 0 || window < 0 || (window & 1)) return ANON_ERR_INVALID_ARG;
    WsCursor ws = ws_begin(ctx);
    AttnPlan plan;
    int rc = attention_plan(ctx, ws, h_cu_seqlens, B, dtype, &plan, window);
    if (rc) return rc;
    return attention_run(ctx, plan, d_qkv, d_cu_seqlens, h_cu_seqlens[0], B, hidden, heads, dtype, d_ctx);
}

#if ATT_PROF
extern "C" int anon_debug_att_prof(unsigned long long* out) { return (int)cudaMemcpyFromSymbol(out, g_att_prof, sizeof(unsigned long long) * 64); }
#endif
