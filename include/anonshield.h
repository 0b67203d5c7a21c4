/*
 * anonshield.h -- C ABI of the B200-native AnonShield pseudonymization hot path
 * (arxiv/paper_2606_15650).  Every entry point is plain C: pointers + sizes, no C++ or
 * torch types.  `d_*` arguments are DEVICE pointers owned by the caller (allocated e.g.
 * through PyTorch); `h_*` / un-prefixed pointers are HOST pointers.  The library never
 * frees caller memory and keeps no caller pointer after a call returns, except inside
 * handles it created (anon_weights keeps its own device copy of the parameters,
 * anon_cache copies entity bytes into its own arena).
 *
 * Citations: P:L<n> = /root/reference/PAPER.md line n; BJ = BASELINE.json north_star;
 * S8x = SURVEY.md section 8(x); Dn = DESIGN.md reading n.
 *
 * Execution model.  All work is enqueued on the cudaStream_t given to anon_ctx_create.
 * Calls are asynchronous with respect to the host unless stated ("synchronises").
 * Device-side failures that are only known after kernels ran (span list / arena
 * capacity, table full) are latched in a sticky per-context status word that
 * anon_ctx_sync() returns and clears.  No exception or abort crosses the ABI.  One
 * context per host thread; handles are not thread-safe.  There is NO CPU fallback: on a
 * machine without a CUDA device every compute call returns ANON_ERR_CUDA.
 */
#ifndef ANONSHIELD_H
#define ANONSHIELD_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* ---- return codes -------------------------------------------------------------------- */
#define ANON_OK                 0
#define ANON_ERR_INVALID_ARG   -1   /* NULL where a pointer is required, negative size ...        */
#define ANON_ERR_UNSUPPORTED   -2   /* d_head != 64, n_i > max_pos, even num_labels, S >= 2^31 ... */
#define ANON_ERR_CAPACITY      -3   /* span list / cache / arena / output buffer too small; the   */
                                    /* needed count is still written where the call documents it  */
#define ANON_ERR_KEY_MISMATCH  -4   /* cache already bound to another HMAC key                    */
#define ANON_ERR_CUDA          -5   /* CUDA runtime error; see anon_last_cuda_error               */
#define ANON_ERR_OOM           -6   /* workspace or device allocation too small / failed          */

typedef struct anon_ctx     anon_ctx;
typedef struct anon_weights anon_weights;
typedef struct anon_cache   anon_cache;
typedef struct anon_regex   anon_regex;

/* Encoder shape (BJ "embedding plus L encoder layers ... then the token-classification
 * head"; S8c O1).  dtype: 0 = FP32 parameters and arithmetic (BJ configs[0]);
 * 1 = BF16 matrices/embeddings, FP32 accumulate, FP32 residual stream / LayerNorm /
 * softmax / logits (BJ configs[1..3], S8c reading S8). */
typedef struct {
    int32_t layers, hidden, heads, ffn, vocab, num_labels, max_pos;
    float   ln_eps;
    int32_t dtype;
    /* S8f NEXT-3, reading D20.  arch 0 (all further fields ignored) = the post-LN BERT-style block above; arch 1 = the
     * ModernBERT-shaped block: pre-LN without bias terms, rotary position embedding on q and k (rotate-half pairing,
     * angle = pos * theta^(-2i/64)), GeGLU feed-forward (W_i is [2 ffn, hidden]: gelu(first half) * second half), no
     * biases except b_c; layer l attends globally (rope_theta_global) iff l % global_every == 0, else only to keys with
     * |i - j| <= local_window / 2 (rope_theta_local).  dtype 1 supports local_window = 128 (or no local layer). */
    int32_t arch, local_window, global_every;
    float   rope_theta_global, rope_theta_local;
} anon_model_desc;

/* Per-token metadata for span decoding (S8c O3).  flags bit0 = keep. */
typedef struct { int32_t record_id, char_start, char_end, flags; } anon_tok_meta;
/* One decoded entity span: bytes [char_start, char_end) of record record_id. */
typedef struct { int32_t record_id, char_start, char_end, type; } anon_span;

const char* anon_strerror(int code);
/* Name of every exported entry point, NULL-terminated (used by the load/export test). */
const char* const* anon_exported_symbols(void);

/* ---- context --------------------------------------------------------------------------- */
/* Creates a context on CUDA device `device` that enqueues on `cuda_stream` (a cudaStream_t
 * passed as void*; NULL = the legacy default stream) and owns a scratch workspace of
 * `workspace_bytes` bytes of device memory (0 is legal: calls that need scratch then
 * return ANON_ERR_OOM).  Synchronises.  Errors: INVALID_ARG, CUDA, OOM. */
int  anon_ctx_create(anon_ctx** out, int device, void* cuda_stream, size_t workspace_bytes);
void anon_ctx_destroy(anon_ctx* ctx);
/* Waits for the context's stream; returns and clears the sticky device status (ANON_OK,
 * ANON_ERR_CAPACITY, ANON_ERR_UNSUPPORTED or ANON_ERR_CUDA). */
int  anon_ctx_sync(anon_ctx* ctx);
/* Text of the last CUDA error seen by this context ("" if none).  Owned by the context. */
const char* anon_last_cuda_error(anon_ctx* ctx);
/* Launch accounting and per-kernel-class CUDA-event timing (bench.py's roofline / gpu_launches keys).
 * anon_ctx_profile(ctx, 1) synchronises, zeroes the counters and starts bracketing every launch group
 * with events on the context stream; (ctx, 0) stops.  anon_ctx_profile_read synchronises and returns,
 * for class c (0 = QKV GEMM, 1 = attention, 2 = row kernels embed/LN/head, 3 = decode+gather+splice,
 * 4 = pseudonymize, 5 = out-projection GEMM, 6 = FFN1+GELU GEMM, 7 = FFN2 GEMM; arrays of 8): summed event time in ms, algorithmic work (FLOPs for classes 0-1
 * and 5-7, bytes for 2-3, 0 for 4), launches; and the total number of kernels launched since the last
 * anon_ctx_profile call (counted whether or not timing is enabled).  Any pointer may be NULL. */
int  anon_ctx_profile(anon_ctx* ctx, int enable);
int  anon_ctx_profile_read(anon_ctx* ctx, double* class_ms, double* class_work, int64_t* class_launches,
                           int64_t* total_launches);
/* Scratch bytes anon_ner_forward needs to process `max_tokens` packed tokens in
 * `max_seqs` sequences in ONE pass; with less, anon_ner_forward splits the batch into
 * sequence-aligned chunks that fit (at least one 512-token sequence must fit).  Also
 * covers anon_decode_spans / anon_gather_spans / anon_pseudonymize for max_tokens items. */
size_t anon_workspace_bytes(const anon_model_desc* desc, int64_t max_tokens, int32_t max_seqs);

/* ---- parameters -------------------------------------------------------------------------- */
/* Uploads the parameters.  `host_fp32_blob` holds n_floats FP32 values in the fixed order
 *   E_w[V,H], E_p[max_pos,H], E_t[H], g_e[H], b_e[H],
 *   { W_qkv[3H,H], b_qkv[3H], W_o[H,H], b_o[H], g_1[H], b_1[H],
 *     W_1[F,H], b_1f[F], W_2[H,F], b_2f[H], g_2[H], b_2[H] } x layers,
 *   W_c[NL,H], b_c[NL]
 * (all matrices row-major [out,in]: y = W x + b; S8d W0).  For arch 1 the order is
 *   E_w[V,H], g_e[H], { g_a[H], W_qkv[3H,H], W_o[H,H], g_m[H], W_i[2F,H], W_2[H,F] } x layers, g_f[H], W_c[NL,H], b_c[NL].  For dtype 1 the matrices and
 * embedding tables are converted to BF16 (round-to-nearest-even; exact when the caller
 * pre-rounded them).  Synchronises.  Errors: INVALID_ARG (size mismatch), UNSUPPORTED
 * (hidden/heads != 64, hidden % 64, ffn % 64, even num_labels, num_labels > 64,
 * max_pos > 512), CUDA, OOM. */
int  anon_weights_load(anon_ctx* ctx, const anon_model_desc* desc, const float* host_fp32_blob,
                       size_t n_floats, anon_weights** out);
void anon_weights_free(anon_weights* w);

/* ---- A1-A8: encoder forward + head + argmax (BJ ¶1; S8c O1, O2) ---------------------- */
/* d_token_ids int32[T] packed, d_cu_seqlens int32[B+1] with [0]=0, [B]=T, every length in
 * [0, max_pos].  Position ids are 0..n_i-1 inside each sequence; attention spans exactly
 * the tokens of the same sequence (bidirectional).  Writes logits FP32 [T, num_labels]
 * row-major if d_logits != NULL and labels int32[T] (argmax, ties -> lowest index, taken on
 * the FP32 logits) if d_labels != NULL.  Reads d_cu_seqlens on the host (one small D2H
 * copy + stream sync at entry) to plan chunks and attention work.  Errors: INVALID_ARG,
 * UNSUPPORTED (a sequence longer than max_pos, token id outside [0,V) is clamped and
 * latches UNSUPPORTED in the sticky status), OOM (workspace cannot hold one sequence), CUDA. */
int  anon_ner_forward(anon_ctx* ctx, const anon_weights* w,
                      const int32_t* d_token_ids, const int32_t* d_cu_seqlens, int32_t B, int32_t T,
                      float* d_logits, int32_t* d_labels);

/* ---- A9: BIO decode + stream compaction (BJ ¶1; S8c O3) -------------------------------------- */
/* Label map 0 = O, 2t+1 = B-t, 2t+2 = I-t.  Tokens with keep = 0 are transparent.  Spans are
 * written in order of their first token.  *d_num_spans (device int32) receives the TOTAL
 * number of spans found even when it exceeds span_capacity; only the first span_capacity
 * are written and ANON_ERR_CAPACITY is latched in the sticky status.  Asynchronous. */
int  anon_decode_spans(anon_ctx* ctx, const int32_t* d_labels, const anon_tok_meta* d_meta, int32_t T,
                       int32_t num_labels, anon_span* d_spans, int32_t span_capacity, int32_t* d_num_spans);

/* A9 for callers that may not allocate (code under CUDA graph capture, serving loops, harnesses that forbid cudaMalloc): the
 * same decode, same kernels and same results as anon_decode_spans, but it needs no context and no workspace.  Its scratch
 * (previous-kept-token index per token, the scan aggregates, a status word; 4.2 MB) is a file-scope device array inside the
 * library that every GPU loading the library holds until exit.  The call allocates nothing: kernel launches and one 4-byte
 * memset on `cuda_stream` (NULL = the default stream) of `device`, which it makes current.  Asynchronous.
 * Limit: T <= ANON_DECODE_STATIC_MAX_TOKENS, else ANON_ERR_CAPACITY and nothing is launched (use anon_decode_spans).
 * All calls on one device share the array: calls that overlap on the GPU (different streams without an ordering between them)
 * race and give undefined spans -- keep them stream-ordered.  The array keeps the last call's contents; each call rewrites what
 * it reads and clears the status word, so nothing carries over.  There is no sticky status here: span_capacity overflow is
 * reported only through *d_num_spans > span_capacity (the first span_capacity spans are written, as in anon_decode_spans).
 * All pointers are device pointers owned by the caller.  Errors: INVALID_ARG, UNSUPPORTED (num_labels even or < 1), CAPACITY
 * (T beyond the limit), CUDA. */
#define ANON_DECODE_STATIC_MAX_TOKENS 1048576
int  anon_decode_spans_static(int device, void* cuda_stream, const int32_t* d_labels, const anon_tok_meta* d_meta, int32_t T,
                              int32_t num_labels, anon_span* d_spans, int32_t span_capacity, int32_t* d_num_spans);

/* ---- A10: span byte gather (S8a A10) ---------------------------------------------------------- */
/* span_bytes[off_s : off_s + len_s] = text[rec_off[record_id] + char_start : ... + char_end],
 * d_span_offsets int64[S+1] = exclusive prefix sum of the lengths; d_span_type uint8[S]
 * (optional) receives spans[s].type.  If the total exceeds bytes_capacity nothing beyond it
 * is written and ANON_ERR_CAPACITY is latched.  Asynchronous. */
int  anon_gather_spans(anon_ctx* ctx, const uint8_t* d_text, const int64_t* d_record_offsets,
                       const anon_span* d_spans, int32_t S,
                       uint8_t* d_span_bytes, size_t bytes_capacity, int64_t* d_span_offsets,
                       uint8_t* d_span_type);

/* ---- A11-A13: hash-cache dedup, HMAC-SHA256, pseudonym write-back (S8c O4) */
/* An open-addressing table with room for max_unique distinct entity strings (slots =
 * next power of two >= 2*max_unique) plus an arena of key_arena_bytes for their bytes and
 * 32 bytes of digest each.  Nothing is evicted implicitly (reading S18); anon_cache_evict shrinks it on request.  Synchronises. */
int  anon_cache_create(anon_ctx* ctx, uint64_t max_unique, uint64_t key_arena_bytes, anon_cache** out);
void anon_cache_destroy(anon_cache* c);
/* Forgets every entry, the counters and the key binding (table memset on the context stream;
 * arena and digests are simply reused).  Asynchronous.  bench.py calls it between steps so that
 * every step inserts and HMACs the same set of new entities. */
int  anon_cache_clear(anon_cache* c);
/* Counters since creation (or the last anon_cache_clear).  Synchronises. */
int  anon_cache_stats(anon_cache* c, uint64_t* n_unique, uint64_t* n_lookups, uint64_t* n_hits);
/* Entry `uid` (0 <= uid < n_unique): copies min(len, bytes_capacity) entity bytes to
 * h_bytes (may be NULL), the 32-byte digest to h_digest (may be NULL); returns the entity
 * length or a negative error.  Synchronises.  (The (entity, slug, full_hash) hand-off
 * of P:L52.) */
int64_t anon_cache_entry(anon_cache* c, uint64_t uid, uint8_t* h_bytes, size_t bytes_capacity,
                         uint8_t* h_digest);

/* The whole mapping table at once, in uid (first-occurrence) order: entity bytes as CSR (h_bytes, h_offsets
 * int64[n_unique + 1]) and the 32-byte digests -- the (original_name, full_hash) columns of the paper's SQLite
 * mapping; slug_name is the first slug_len hex characters of the digest, entity_type travels with the spans.
 * Any output pointer may be NULL; *n_unique / *n_bytes are always written, so a first call with NULL buffers sizes
 * the second.  ANON_ERR_CAPACITY if bytes_capacity is too small.  Re-inserting the exported entities in this order
 * into a fresh cache (anon_pseudonymize with the same key) reproduces the same uids and digests (resume).
 * Synchronises. */
int  anon_cache_export(anon_cache* c, uint8_t* h_bytes, size_t bytes_capacity, int64_t* h_offsets, uint8_t* h_digests,
                       uint64_t* n_unique, uint64_t* n_bytes);

/* ---- NEXT-5: bounded cache, call-granular LRU eviction ("LRU cache"; S8f NEXT-5; reading D21) ------------------------ */
/* Enables (or with 0 disables and forgets) recency tracking: from now on every anon_pseudonymize call stamps each entry it
 * looks up -- hit or newly inserted -- with the call's sequence number (4 bytes of device memory per max_unique; entries that
 * predate tracking count as oldest).  Synchronises.  Errors: OOM, CUDA. */
int  anon_cache_track_use(anon_cache* c, int enable);
/* Shrinks the cache to its `keep` most recently used entries: the entries with the largest stamps stay, inside the cut-off
 * stamp the lowest uids stay; everything else is forgotten (a later lookup of such a string is a miss and recomputes the
 * same HMAC -- no pseudonym ever changes).  Survivors are renumbered 0..keep-1 in their old uid order and keep their
 * bytes, digests and stamps; the lookup / hit counters and the key binding are untouched.  Export the mapping
 * (anon_cache_export) BEFORE evicting if it must stay complete (the paper's persistent mapping).  keep >= n_unique is
 * a no-op.  *n_evicted (may be NULL) receives the number of entries dropped.  Needs workspace for the surviving bytes plus
 * 45 bytes per entry.  Synchronises.  Errors: UNSUPPORTED (tracking not enabled), OOM, CUDA. */
int  anon_cache_evict(anon_cache* c, uint64_t keep, uint64_t* n_evicted);

/* For span i = 0..S-1 in order (e_i = d_span_bytes[off[i] .. off[i+1]), exact bytes):
 *   hit[i] = 1 if e_i is already in the cache (from an earlier call or an earlier i), else 0
 *            and (HMAC_SHA256(key, e_i), uid = number of entries before insertion) is inserted;
 *   uid[i] = uid of e_i;  digests[i] = its 32-byte HMAC;
 *   out[i] = "[" type_names[type[i]] "_" lowerhex(digest)[0:slug_len] "]"   (type 0 if d_span_type NULL);
 *   d_out_offsets int64[S+1] = exclusive prefix sum of the token lengths.
 * key: HOST pointer, any length (keys > 64 bytes are hashed first, RFC 2104).  The cache
 * binds to the first key it sees; another key -> ANON_ERR_KEY_MISMATCH.  slug_len in
 * [0,64].  type_names: HOST array of num_types NUL-terminated ASCII names (<= 32 bytes
 * each, num_types <= 64); a type >= num_types is clamped to num_types-1 and latches
 * ANON_ERR_UNSUPPORTED in the sticky status.  d_hit / d_uid / d_digests may be NULL.
 * Alignment: d_span_offsets / d_out_offsets / d_uid are int64 arrays (8-byte aligned); d_digests, when given, must be
 * 16-byte aligned (ANON_ERR_INVALID_ARG otherwise); d_span_bytes, d_out_tokens, d_span_type and d_hit may sit at ANY byte
 * address (e.g. a sub-buffer of a larger allocation).  S > 0 needs d_span_bytes and d_out_tokens (INVALID_ARG if NULL).
 * Synchronises once (to learn how many entities are new, so that capacity errors are
 * returned, not latched): on ANON_ERR_CAPACITY (max_unique, arena or out_capacity
 * exceeded) the cache is left exactly as before the call.  S must be < 2^31.
 * Workspace: 9 S + 24 (S / 2048 + 2) bytes plus alignment (ANON_ERR_OOM if the context has less). */
int  anon_pseudonymize(anon_ctx* ctx, anon_cache* cache,
                       const uint8_t* d_span_bytes, const int64_t* d_span_offsets,
                       const uint8_t* d_span_type, int64_t S,
                       const uint8_t* key, size_t key_len, int32_t slug_len,
                       const char* const* type_names, int32_t num_types,
                       uint8_t* d_out_tokens, size_t out_capacity, int64_t* d_out_offsets,
                       uint8_t* d_hit, int64_t* d_uid, uint8_t* d_digests);

/* A12 alone, dedup disabled: digests[i] = HMAC_SHA256(key, e_i) for every span (used to
 * measure the SHA-256 kernel's integer issue rate, S8d c5).  Asynchronous.  d_digests must be
 * 16-byte aligned (ANON_ERR_INVALID_ARG otherwise); d_span_bytes may sit at any byte address. */
int  anon_hmac_spans(anon_ctx* ctx, const uint8_t* d_span_bytes, const int64_t* d_span_offsets, int64_t S,
                     const uint8_t* key, size_t key_len, uint8_t* d_digests /* [S,32] */);

/* ---- LayerNorm folded into the GEMMs around it (S8a A4 / A6 -> A2; DESIGN.md section 6 "fold") ---------------------------
 * The LayerNorm between a layer's FFN and the next layer's QKV projection does not run as a kernel in the BF16 encoder
 * (hidden 768 / 1024): the FFN2 GEMM (producer) also writes the BF16 copy of its un-normalised output rows and, per row and
 * per 256-column tile, the partial (sum, sum of squares); the QKV GEMM (consumer) multiplies the raw BF16 rows by
 * Wf = bf16(W * gamma) and finishes the LayerNorm in its epilogue.  Both are exposed for parity tests and measurements.
 * Row statistics: part float[M][N_stat / 256][2]; mean = sum / N_stat, rstd = 1 / sqrt(sumsq / N_stat - mean^2 + eps). */
/* Producer: C[M,N] FP32 = A[M,K] W[N,K]^T + bias + R, Cb = bf16(C), part_out[M][N/256][2] = partial sums of C, where
 * R = d_res if both d_res_part and d_res_stats are NULL, else R = LN(d_res; gamma, beta) with the rows' (mean, rstd) taken
 * from d_res_part (partial sums, layout above with N_stat = N) or from d_res_stats (float [M][2] = mean, rstd); giving both
 * is INVALID_ARG.  N in {256, 512, 768, 1024}, K % 64 == 0 (else UNSUPPORTED).  d_C may alias d_res.  Asynchronous. */
int  anon_gemm_bf16_fold_res(anon_ctx* ctx, const void* d_A, const void* d_W, const float* d_bias, const float* d_res,
                             const float* d_res_part, const float* d_res_stats, const float* d_gamma, const float* d_beta,
                             float eps, float* d_C, void* d_Cb, float* d_part_out, int32_t M, int32_t N, int32_t K);
/* Consumer: C[M,N] BF16 = rstd_r * (A_raw[M,K] Wf[N,K]^T - mean_r * s[n]) + c[n], i.e. LN(A_raw; gamma, beta) W^T + b when
 * Wf = bf16(W * gamma), s[n] = sum_k Wf[n,k], c[n] = b[n] + sum_k beta[k] W[n,k]; (mean_r, rstd_r) from d_part with
 * N_stat = stat_cols (a multiple of 256, normally K).  N > 128, N % 8 == 0, K % 64 == 0.  Asynchronous. */
int  anon_gemm_bf16_fold(anon_ctx* ctx, const void* d_A_raw, const void* d_Wf, const float* d_c, const float* d_s,
                         const float* d_part, int32_t stat_cols, float eps, void* d_C, int32_t M, int32_t N, int32_t K);

/* ---- measured issue-rate peaks ("Integer-ALU and MUFU rates are not in MEASURED_PEAKS.json --
 * measure"): the denominators of the "alu" roofline of HMAC-SHA256 (K10) and of the exp ceiling of attention (K3). -------------- */
/* Runs a register-only micro-kernel (2,048 resident threads per SM, 8 independent chains per thread, no memory traffic in the
 * timed loop) and returns thread-level operations per second (= lanes/clk/SM x SMs x clock) in *thread_ops_per_s, best of three
 * launches timed with CUDA events on the context stream; *kernel_ms (may be NULL) = that launch's duration.
 * mode 0: LOP3 + funnel shift + three-input add per step (the SHA-256 mix; ptxas spreads it over the ALU and FMA pipes: LOP3 +
 * LEA.HI + IMAD.IADD, counted as 3 operations); 1: LOP3 only; 2: SHF only; 3: IADD3 only; 4: MUFU ex2.approx only.
 * iters in [1, 2^20]: outer loop trips, 128 operations (x3 in mode 0) per thread and trip.  Synchronises.
 * Errors: INVALID_ARG, CUDA. */
int  anon_microbench(anon_ctx* ctx, int32_t mode, int32_t iters, double* thread_ops_per_s, double* kernel_ms);

/* ---- NEXT-1: record splice (P:L53 stage 5 restricted to record text; S8f NEXT-1) ------------------------------- */
/* Rewrites every record with each span [char_start, char_end) replaced by its pseudonym token:
 *   new_text = for each record, the bytes between spans copied, out_tokens[out_offsets[s] .. out_offsets[s+1]) in
 *   place of span s;  d_new_record_offsets int64[R+1] = offsets of the rewritten records.
 * d_spans must be in stream order (as anon_decode_spans writes them) and non-overlapping; text_bytes =
 * record_offsets[R].  If the rewritten text exceeds new_text_capacity nothing beyond it is written and
 * ANON_ERR_CAPACITY is latched in the sticky status.  Workspace: 16 (S + 1) + new_text_capacity / 1024 + 64 KB bytes
 * (ANON_ERR_OOM if the context has less).  d_text, d_out_tokens and d_new_text may sit at any byte address.  Asynchronous. */
int  anon_splice_records(anon_ctx* ctx, const uint8_t* d_text, size_t text_bytes, const int64_t* d_record_offsets, int32_t R,
                         const anon_span* d_spans, int32_t S, const uint8_t* d_out_tokens, const int64_t* d_out_offsets,
                         uint8_t* d_new_text, size_t new_text_capacity, int64_t* d_new_record_offsets);

/* ---- NEXT-4: regex detector and regex / NER span merge ("custom regex patterns"; S8f NEXT-4; D17-D19) ----- */
/* Uploads a pattern automaton.  h_blob (HOST pointer) is a deterministic finite automaton over byte classes for ALL patterns
 * at once; paper_2606_15650_b200/regex_dfa.py compile_patterns() builds it from a restricted regex syntax, and any other
 * producer (a C caller with its own DFA) may write the same bytes.  Layout, little-endian, no padding except where stated:
 *   uint32 head[8]      = { 0x31585241 ("ARX1"), n_states (2..65535), n_classes (1..128), n_patterns (1..127),
 *                           max_match (1..255 bytes), 0, 0, 0 }
 *   uint8  class_of[256]   byte value -> class index (< n_classes)
 *   uint8  is_word[256]    1 if the byte is a word character ([0-9A-Za-z_], rule D18's boundary test), else 0
 *   uint8  type_of[256]    pattern index -> span type written into anon_span.type (entries >= n_patterns unused)
 *   int16  accept[n_states]   pattern index accepted in this state (lowest index if several), -1 if none;
 *                             zero-padded to a multiple of 4 bytes
 *   uint16 trans[n_states][n_classes]   next state
 * State 0 is the dead state (all its transitions are 0, it accepts nothing), state 1 the start state (must not accept: no
 * empty match).  blob_bytes must equal 32 + 768 + round4(2 n_states) + 2 n_states n_classes.  The tables are validated here (sizes, every transition and
 * accept label in range, at most 127 patterns, max_match <= 255) and must fit shared memory beside a text tile, else
 * ANON_ERR_UNSUPPORTED.  The handle keeps its own device copy.  Synchronises.  Errors: INVALID_ARG, UNSUPPORTED, OOM, CUDA. */
int  anon_regex_load(anon_ctx* ctx, const void* h_blob, size_t blob_bytes, anon_regex** out);
void anon_regex_free(anon_regex* rx);
/* Scans every record for the patterns, rule D18: matches are taken left to right inside a record, never overlap and never
 * cross a record boundary; at a position the longest match wins (at most max_match bytes), ties go to the lowest pattern
 * index; a match starts and ends at a word boundary (the byte before / after is not [0-9A-Za-z_], or it is the record's
 * edge).  d_record_offsets int64[R+1] with [0] = 0 and [R] = text_bytes.  Spans are written in stream order
 * (record, char_start) with type = type_of_pattern[pattern]; *d_num_spans (device) receives the TOTAL found, only the
 * first span_capacity are written and ANON_ERR_CAPACITY is latched beyond.  Workspace: 2 * text_bytes + 12 * R + small.
 * Asynchronous. */
int  anon_regex_scan(anon_ctx* ctx, const anon_regex* rx, const uint8_t* d_text, size_t text_bytes,
                     const int64_t* d_record_offsets, int32_t R, anon_span* d_spans, int32_t span_capacity,
                     int32_t* d_num_spans);
/* Rule D19: every regex span is kept; an NER span is kept iff it overlaps no regex span of its record; the result is
 * ordered by (record_id, char_start), an NER span before a regex span on a tie.  Both inputs must be ordered by
 * (record_id, char_start) and the regex spans non-overlapping (anon_decode_spans and anon_regex_scan write them so).
 * The counts may live on the device: d_num_ner / d_num_regex (device int32, clamped to *_max) or NULL = *_max itself.
 * *d_num_out (device) receives the merged count even when it exceeds `capacity` (then ANON_ERR_CAPACITY is latched).
 * d_out_spans must not alias an input.  Asynchronous. */
int  anon_merge_spans(anon_ctx* ctx, const anon_span* d_ner_spans, const int32_t* d_num_ner, int32_t ner_max,
                      const anon_span* d_regex_spans, const int32_t* d_num_regex, int32_t regex_max,
                      anon_span* d_out_spans, int32_t capacity, int32_t* d_num_out);
/* Attaches a pattern automaton to the context (NULL detaches): anon_pipeline_host / anon_pipeline_host_text then run
 * anon_regex_scan on the batch text and anon_merge_spans between the BIO decode and the span gather, so the spans they
 * return, pseudonymize and splice are the merged list (the paper's hybrid strategy).  The handle must outlive its
 * attachment.  The regex types index the same type_names array as the NER types. */
int  anon_ctx_set_regex(anon_ctx* ctx, const anon_regex* rx);

/* ---- whole hot path with HOST buffers (the call a user makes; bench.py's e2e leg) ------------- */
/* Copies one batch host->device, runs A1-A13 and copies the results back, all on the
 * context's stream; synchronises before returning.  Host inputs: token_ids int32[T],
 * cu_seqlens int32[B+1], meta[T], text uint8[text_bytes], record_offsets int64[R+1].
 * Host outputs: spans[span_capacity], *num_spans, out_tokens[out_capacity],
 * out_offsets int64[span_capacity+1], hit uint8[span_capacity] (may be NULL).
 * Device staging comes from the context workspace (ANON_ERR_OOM if too small).  Returns
 * ANON_ERR_CAPACITY (with *num_spans = needed) if the span list or outputs do not fit. */
int  anon_pipeline_host(anon_ctx* ctx, const anon_weights* w, anon_cache* cache,
                        const int32_t* h_token_ids, const int32_t* h_cu_seqlens, int32_t B, int32_t T,
                        const anon_tok_meta* h_meta, const uint8_t* h_text, size_t text_bytes,
                        const int64_t* h_record_offsets, int32_t R,
                        const uint8_t* key, size_t key_len, int32_t slug_len,
                        const char* const* type_names, int32_t num_types,
                        anon_span* h_spans, int32_t span_capacity, int32_t* h_num_spans,
                        uint8_t* h_out_tokens, size_t out_capacity, int64_t* h_out_offsets,
                        uint8_t* h_hit);

/* Same, and the records come back REWRITTEN (stage 5 of the paper's pipeline, restricted to record text): after
 * anon_pseudonymize the device splices every token over its span (anon_splice_records) and copies the new text
 * (h_new_record_offsets[R] bytes) and its int64[R+1] record offsets to the host.  new_text_capacity must be at least
 * text_bytes + the total token bytes (text_bytes + out_capacity always suffices), else ANON_ERR_CAPACITY. */
int  anon_pipeline_host_text(anon_ctx* ctx, const anon_weights* w, anon_cache* cache,
                             const int32_t* h_token_ids, const int32_t* h_cu_seqlens, int32_t B, int32_t T,
                             const anon_tok_meta* h_meta, const uint8_t* h_text, size_t text_bytes,
                             const int64_t* h_record_offsets, int32_t R,
                             const uint8_t* key, size_t key_len, int32_t slug_len,
                             const char* const* type_names, int32_t num_types,
                             anon_span* h_spans, int32_t span_capacity, int32_t* h_num_spans,
                             uint8_t* h_out_tokens, size_t out_capacity, int64_t* h_out_offsets,
                             uint8_t* h_hit,
                             uint8_t* h_new_text, size_t new_text_capacity, int64_t* h_new_record_offsets);

/* ---- building blocks exported for parity tests and per-kernel roofline measurement ----------- */
/* C[M,N] = A[M,K] * W[N,K]^T + bias[N], BF16 operands, FP32 accumulate on the tcgen05
 * tensor cores (S8a A2/A4/A5/A6).  epilogue: 0 = bias -> BF16 out; 1 = bias, erf-GELU ->
 * BF16 out; 2 = bias + FP32 residual[M,N] -> FP32 out; 4 = GeGLU (NEXT-3): C is BF16 [M, N/2] with
 * C[:, 128t + j] = gelu(acc[:, 256t + j]) * acc[:, 256t + 128 + j], i.e. W holds, per 256-row tile, 128 "input" rows followed
 * by their 128 gate rows; no bias is added; N % 256 == 0.  K % 64 == 0, N % 8 == 0 required.
 * d_A, d_W BF16 (uint16 bit patterns) row-major, 16-byte aligned.  Asynchronous. */
int  anon_gemm_bf16(anon_ctx* ctx, const void* d_A, const void* d_W, const float* d_bias,
                    const float* d_residual, void* d_C, int32_t M, int32_t N, int32_t K, int32_t epilogue);
/* ctx[T,H] = varlen bidirectional softmax attention over qkv[T,3H] (S8a A3); dtype as in
 * anon_model_desc (0: FP32 qkv/ctx, 1: BF16).  h_cu_seqlens is a HOST pointer.  Asynchronous. */
int  anon_attention(anon_ctx* ctx, const void* d_qkv, const int32_t* d_cu_seqlens,
                    const int32_t* h_cu_seqlens, int32_t B, int32_t T, int32_t hidden, int32_t heads,
                    int32_t dtype, void* d_ctx);
/* Same with a local window (NEXT-3, D20): query i sees the keys j of its sequence with |i - j| <= window / 2; window 0 =
 * anon_attention.  dtype 1 supports window 128 only (ANON_ERR_UNSUPPORTED otherwise).  Asynchronous. */
int  anon_attention_local(anon_ctx* ctx, const void* d_qkv, const int32_t* d_cu_seqlens,
                          const int32_t* h_cu_seqlens, int32_t B, int32_t T, int32_t hidden, int32_t heads,
                          int32_t dtype, int32_t window, void* d_ctx);

#ifdef __cplusplus
}
#endif
#endif /* ANONSHIELD_H */
