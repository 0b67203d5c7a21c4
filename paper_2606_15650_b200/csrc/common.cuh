// common.cuh -- context, error plumbing and workspace cursor shared by the translation units of
// libanonshield.so (product code; shares nothing with oracle/).
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <cuda_bf16.h>
#include <stdint.h>
#include <stddef.h>
#include <stdio.h>
#include <string.h>
#include <vector>

#include "../../include/anonshield.h"

// per-kernel-class CUDA-event timing (anon_ctx_profile): classes index ctx->prof_* arrays
// PROF_GEMM = QKV projection (bias epilogue); the other three GEMMs have classes of their own so that bench.py can put
// the single dominant kernel against its roofline
enum ProfClass { PROF_GEMM = 0, PROF_ATTN = 1, PROF_ROW = 2, PROF_DECODE = 3, PROF_PSEUDO = 4, PROF_GEMM_OUT = 5,
                 PROF_GEMM_FFN1 = 6, PROF_GEMM_FFN2 = 7, PROF_NCLASS = 8 };
struct ProfRec { cudaEvent_t a, b; int cls; };

struct anon_ctx {
    int device = 0;
    cudaStream_t stream = nullptr;
    uint8_t* ws = nullptr;          // device scratch
    size_t ws_bytes = 0;
    int* d_status = nullptr;        // sticky device-side status word (0 = ok, else first ANON_ERR_*); 256-byte allocation:
                                    // word 16 = the cache probe's own "table full" flag (zeroed by every anon_pseudonymize)
    uint8_t* h_pinned = nullptr;    // small pinned host buffer for read-backs
    size_t h_pinned_bytes = 0;
    int sm_count = 148;
    char cuda_err[256] = {0};
    // cached driver entry point for cuTensorMapEncodeTiled (resolved lazily, see gemm_tcgen05.cu)
    void* encode_tiled = nullptr;
    int smem_optin = 0;
    // tensor maps already encoded for this context (the same activation / weight buffers come back every layer and every step):
    // make_tmap_2d looks here before calling cuTensorMapEncodeTiled
    struct TmapKey { const void* base; uint64_t rows, cols; uint32_t box_cols, box_rows, dt; };
    std::vector<TmapKey> tmap_keys;
    std::vector<CUtensorMap> tmap_vals;
    // kernels whose MaxDynamicSharedMemorySize opt-in has been set on THIS context's device (the attribute is per device)
    const void* smem_attr_done[48] = {nullptr};
    int n_smem_attr_done = 0;
    long long chunk_tokens_cap = 0;     // ANON_CHUNK_TOKENS read once at context creation (0 = workspace-limited only)
    int fold_ln = 1;                    // ANON_FOLD_LN=0 switches the LayerNorm fold off (A/B measurements)
    int ablate = 0;                     // ANON_ABLATE (measurement aid, results are then WRONG): bit 0 skip attention, 1 skip LayerNorm
                                        // kernels, 2 skip the out-projection, 3 FFN1 without GELU -- marginal cost of a kernel class in the step
    // NEXT-4: pattern automaton the host pipeline merges into the NER spans (anon_ctx_set_regex; not owned)
    const struct anon_regex* regex = nullptr;
    // launch accounting + optional event profiling
    long long n_launches = 0;
    bool prof_on = false;
    std::vector<ProfRec> prof_recs;       // events of the current profiling window (pooled, reused)
    size_t prof_used = 0;
    double prof_work[PROF_NCLASS] = {0};
    long long prof_launches[PROF_NCLASS] = {0};
};

// RAII: brackets the launches of one kernel class with events on the context stream (when profiling is on)
struct ProfScope {
    anon_ctx* c; ProfRec* r = nullptr;
    ProfScope(anon_ctx* ctx, int cls, double work, int launches = 1) : c(ctx) {
        c->n_launches += launches;
        if (!c->prof_on) return;
        if (c->prof_used == c->prof_recs.size()) {
            ProfRec n; n.cls = cls;
            if (cudaEventCreate(&n.a) != cudaSuccess || cudaEventCreate(&n.b) != cudaSuccess) return;
            c->prof_recs.push_back(n);
        }
        r = &c->prof_recs[c->prof_used++];
        r->cls = cls;
        c->prof_work[cls] += work;
        c->prof_launches[cls] += launches;
        cudaEventRecord(r->a, c->stream);
    }
    ~ProfScope() { if (r) cudaEventRecord(r->b, c->stream); }
};

// Bump cursor over the context workspace.  Every public entry point starts one at offset 0
// (stream order makes reuse across calls safe); anon_pipeline_host carves its staging first and
// hands the remainder to the stages.
struct WsCursor {
    uint8_t* base; size_t cap; size_t used;
    __host__ void* take(size_t bytes, size_t align = 256) {
        size_t o = (used + align - 1) / align * align;
        if (o + bytes > cap) return nullptr;
        used = o + bytes;
        return base + o;
    }
    __host__ size_t left() const { return cap > used ? cap - used : 0; }
};
static inline WsCursor ws_begin(anon_ctx* c) { return WsCursor{c->ws, c->ws_bytes, 0}; }

static inline int cuda_fail(anon_ctx* c, cudaError_t e, const char* what) {
    if (c) snprintf(c->cuda_err, sizeof c->cuda_err, "%s: %s", what, cudaGetErrorString(e));
    return ANON_ERR_CUDA;
}
#define CU_TRY(ctx, expr)                                                            \
    do { cudaError_t e__ = (expr); if (e__ != cudaSuccess) return cuda_fail((ctx), e__, #expr); } while (0)
#define CU_LAUNCH_CHECK(ctx, name)                                                   \
    do { cudaError_t e__ = cudaGetLastError(); if (e__ != cudaSuccess) return cuda_fail((ctx), e__, name); } while (0)

// Opt a kernel in to `bytes` of dynamic shared memory on the context's device, once per (context, kernel).
static inline int ensure_smem_attr(anon_ctx* c, const void* func, int bytes) {
    for (int i = 0; i < c->n_smem_attr_done; i++) if (c->smem_attr_done[i] == func) return ANON_OK;
    cudaError_t e = cudaFuncSetAttribute(func, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
    if (e != cudaSuccess) return cuda_fail(c, e, "cudaFuncSetAttribute(MaxDynamicSharedMemorySize)");
    if (c->n_smem_attr_done < 48) c->smem_attr_done[c->n_smem_attr_done++] = func;
    return ANON_OK;
}

__device__ __forceinline__ void latch_status(int* d_status, int code) { atomicCAS(d_status, 0, code); }

static inline int64_t ceil_div64(int64_t a, int64_t b) { return (a + b - 1) / b; }

// ---- internal stage entry points (defined in the per-stage .cu files; all take a cursor) ----
struct anon_weights;
int ner_forward_impl(anon_ctx*, WsCursor&, const anon_weights*, const int32_t* d_ids, const int32_t* d_cu,
                     const int32_t* h_cu, int32_t B, int32_t T, float* d_logits, int32_t* d_labels);
int decode_spans_impl(anon_ctx*, WsCursor&, const int32_t* d_labels, const anon_tok_meta* d_meta, int32_t T,
                      int32_t num_labels, anon_span* d_spans, int32_t cap, int32_t* d_num);
int gather_spans_impl(anon_ctx*, WsCursor&, const uint8_t* d_text, const int64_t* d_rec_off,
                      const anon_span* d_spans, const int32_t* d_num_spans, int32_t S_max,
                      uint8_t* d_bytes, size_t cap, int64_t* d_off, uint8_t* d_type);
int pseudonymize_impl(anon_ctx*, WsCursor&, anon_cache*, const uint8_t* d_bytes, const int64_t* d_off,
                      const uint8_t* d_type, int64_t S, const uint8_t* key, size_t key_len, int32_t slug_len,
                      const char* const* type_names, int32_t num_types, uint8_t* d_out, size_t out_cap,
                      int64_t* d_out_off, uint8_t* d_hit, int64_t* d_uid, uint8_t* d_digests,
                      int64_t* total_out_bytes);
int regex_scan_impl(anon_ctx*, WsCursor&, const anon_regex* rx, const uint8_t* d_text, size_t text_bytes, const int64_t* d_rec_off,
                    int32_t R, anon_span* d_spans, int32_t cap, int32_t* d_num);
int merge_spans_impl(anon_ctx*, WsCursor&, const anon_span* d_ner, const int32_t* d_num_ner, int32_t ner_max, const anon_span* d_rgx,
                     const int32_t* d_num_rgx, int32_t rgx_max, anon_span* d_out, int32_t cap, int32_t* d_num_out);
int gemm_bf16_impl(anon_ctx*, const __nv_bfloat16* A, const __nv_bfloat16* W, const float* bias,
                   const float* residual, void* C, int M, int N, int K, int epilogue);
int gemm_bf16_res_ln_impl(anon_ctx*, const __nv_bfloat16* A, const __nv_bfloat16* W, const float* bias, const float* res_y,
                          const float2* res_stats, const float* gamma, const float* beta, float* C, int M, int N, int K);
// LayerNorm folded into the GEMMs (gemm_tcgen05.cu "FOLD"): producer (residual GEMM that also writes the BF16 raw rows and
// the rows' partial statistics) and consumer (finishes the LayerNorm of its raw A rows in the epilogue)
int gemm_bf16_fold_res_impl(anon_ctx*, const __nv_bfloat16* A, const __nv_bfloat16* W, const float* bias, const float* res_y,
                            const float2* part_in, const float2* res_stats, const float* gamma, const float* beta, float eps, float* C,
                            __nv_bfloat16* Cb, float2* part_out, int M, int N, int K);
int gemm_bf16_fold_impl(anon_ctx*, const __nv_bfloat16* A_raw, const __nv_bfloat16* Wf, const float* c, const float* s_vec,
                        const float2* part_in, int stat_cols, float eps, void* C, int M, int N, int K);
// qkv = A W^T, RoPE on the q / k heads in the epilogue; table float2 [32][512] pair-major (cos, sin), pos int [M]
int gemm_bf16_rope_impl(anon_ctx*, const __nv_bfloat16* A, const __nv_bfloat16* W, const int* pos, const float2* table, void* C,
                        int M, int N, int K);
// 2-D row-major tensor [rows, cols] of esize-byte elements, box [box_rows, box_cols] with box_cols * esize = 128 B,
// 128-byte swizzle (gemm_tcgen05.cu).
int make_tmap_2d(anon_ctx* ctx, CUtensorMap* tm, CUtensorMapDataType dt, uint32_t esize, const void* base, uint64_t rows,
                 uint64_t cols, uint32_t box_cols, uint32_t box_rows);
struct AttnPlan { void* d_work; int n_items; int n_rows; int window; };
// window = 0: every query sees its whole sequence; else keys with |i - j| <= window / 2 (NEXT-3 local layers)
int attention_plan(anon_ctx*, WsCursor&, const int32_t* h_cu, int B, int dtype, AttnPlan* plan, int window = 0);
int attention_run(anon_ctx*, const AttnPlan&, const void* d_qkv, const int32_t* d_cu, int tok0, int B, int hidden,
                  int heads, int dtype, void* d_ctx);
const anon_model_desc* weights_desc(const anon_weights* w);
