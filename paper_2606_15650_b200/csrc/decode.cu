// decode.cu -- A9 BIO span decode + stream compaction (K7) and A10 span byte gather (K8).
// BJ north_star ¶1 ("Per-token argmax and BIO span decoding ... a stream-compacted span list");
// S8c O3 (label map 0=O, 2t+1=B-t, 2t+2=I-t; non-kept tokens transparent; spans break on
// record_id; lenient starts).  Integer work: bit-exact against the oracle.
//
// K7 in two transform-scans over the packed token stream (HBM-bound, 20 B/token read):
//   1. max-scan of (keep ? j : -1)            -> prev_kept[j] = index of the previous kept token
//   2. sum-scan of start(j)                   -> rank of every span start; the apply pass writes
//      (record, char_start, type) at spans[rank] and, for every kept token that does NOT continue
//      its predecessor's span, char_end of spans[rank-1] from that predecessor.  A one-thread
//      fix-up closes the span still open at the end of the stream and publishes the count.
#include "common.cuh"
#include "scan.cuh"

namespace {

struct KeepIn {
    const anon_tok_meta* meta;
    __device__ __forceinline__ int operator()(long long j) const { return (meta[j].flags & 1) ? (int)j : -1; }
};
struct PrevKeptOut {
    int* prev;
    __device__ __forceinline__ void operator()(long long j, int excl, int) const { prev[j] = excl; }
};

__device__ __forceinline__ bool tok_continues(int lab, int rec, int plab, int prec) {
    // O3: j continues iff l_j is an I- label, prev(j) is in the same record, l_prev > 0, same type
    return lab > 0 && (lab & 1) == 0 && plab > 0 && prec == rec && ((plab - 1) >> 1) == ((lab - 1) >> 1);
}

struct StartIn {
    const int* labels; const anon_tok_meta* meta; const int* prev;
    __device__ __forceinline__ long long operator()(long long j) const {
        const anon_tok_meta m = meta[j];
        if (!(m.flags & 1)) return 0;
        const int lab = labels[j];
        if (lab <= 0) return 0;
        const int p = prev[j];
        if (p < 0) return 1;
        return tok_continues(lab, m.record_id, labels[p], meta[p].record_id) ? 0 : 1;
    }
};
struct StartOut {
    const int* labels; const anon_tok_meta* meta; const int* prev; anon_span* spans; long long cap;
    __device__ __forceinline__ void operator()(long long j, long long rank, long long is_start) const {
        const anon_tok_meta m = meta[j];
        if (!(m.flags & 1)) return;
        const int lab = labels[j];
        const int p = prev[j];
        if (is_start && rank < cap) {
            spans[rank].record_id = m.record_id;
            spans[rank].char_start = m.char_start;
            spans[rank].type = (lab - 1) >> 1;
        }
        if (p >= 0) {
            const int plab = labels[p];
            if (plab > 0 && !tok_continues(lab, m.record_id, plab, meta[p].record_id)) {
                // token p was the last token of span rank-1 (rank counts the starts before j)
                if (rank - 1 < cap) spans[rank - 1].char_end = meta[p].char_end;
            }
        }
    }
};

__global__ void decode_finish_kernel(const int* labels, const anon_tok_meta* meta, const int* prev, int T,
                                     const long long* total, anon_span* spans, int cap, int* d_num, int* d_status) {
    const long long n = *total;
    if (T > 0) {
        const int last = (meta[T - 1].flags & 1) ? T - 1 : prev[T - 1];
        if (last >= 0 && labels[last] > 0 && n - 1 < cap) spans[n - 1].char_end = meta[last].char_end;
    }
    *d_num = (int)n;
    if (n > cap) latch_status(d_status, ANON_ERR_CAPACITY);
}

// ---- K8 ----
struct LenIn {
    const anon_span* spans;
    __device__ __forceinline__ long long operator()(long long s) const {
        const int l = spans[s].char_end - spans[s].char_start;
        return l > 0 ? l : 0;
    }
};
struct GatherOut {
    const anon_span* spans; const uint8_t* text; const long long* rec_off;
    uint8_t* out; long long cap; long long* off; uint8_t* type; int* d_status;
    __device__ __forceinline__ void operator()(long long s, long long o, long long len) const {
        off[s] = o;
        const anon_span sp = spans[s];
        if (type) type[s] = (uint8_t)sp.type;
        if (o + len > cap) { latch_status(d_status, ANON_ERR_CAPACITY); return; }
        const uint8_t* src = text + rec_off[sp.record_id] + sp.char_start;
        uint8_t* dst = out + o;
        for (long long k = 0; k < len; k++) dst[k] = src[k];
    }
};
__global__ void gather_finish_kernel(const long long* total, const int* d_n, long long S_max, long long* off) {
    const long long n = d_n ? min((long long)*d_n, S_max) : S_max;
    off[n] = *total;
}

// ---- NEXT-1: record splice (PAPER.md L53 stage 5, restricted to record text) ----
// D[s] = exclusive prefix sum of (token length - span length) over the span list in stream order; a byte at absolute
// position p that lies outside every span moves to p + D[k], k = number of spans that start at or before p; the token
// of span s goes to abs_start[s] + D[s].
struct DeltaIn {
    const anon_span* spans; const long long* tok_off;
    __device__ __forceinline__ long long operator()(long long s) const {
        const int l = spans[s].char_end - spans[s].char_start;
        return (tok_off[s + 1] - tok_off[s]) - (l > 0 ? l : 0);
    }
};
struct DeltaOut {
    const anon_span* spans; const long long* rec_off; long long* D; long long* astart; long long* aend; long long S;
    __device__ __forceinline__ void operator()(long long s, long long ex, long long v) const {
        const anon_span sp = spans[s];
        const long long a = rec_off[sp.record_id] + sp.char_start;
        const int l = sp.char_end - sp.char_start;
        D[s] = ex; astart[s] = a; aend[s] = a + (l > 0 ? l : 0);
        if (s == S - 1) D[S] = ex + v;
    }
};

__global__ void __launch_bounds__(256) splice_copy_kernel(const uint8_t* __restrict__ text, long long nbytes, long long S,
                                                          const long long* __restrict__ D, const long long* __restrict__ astart,
                                                          const long long* __restrict__ aend, uint8_t* __restrict__ out,
                                                          long long cap, int* d_status)
{
    const long long p0 = ((long long)blockIdx.x * blockDim.x + threadIdx.x) * 16;
    if (p0 >= nbytes) return;
    long long lo = 0, hi = S;                       // k = number of spans with astart <= p0
    while (lo < hi) { const long long mid = (lo + hi) >> 1; if (astart[mid] <= p0) lo = mid + 1; else hi = mid; }
    long long k = lo;
    long long prev_end = k > 0 ? aend[k - 1] : -1, next_start = k < S ? astart[k] : nbytes + 16, shift = D[k];
    const long long pe = p0 + 16 < nbytes ? p0 + 16 : nbytes;
    for (long long p = p0; p < pe; p++) {
        while (p >= next_start) { prev_end = aend[k]; k++; next_start = k < S ? astart[k] : nbytes + 16; shift = D[k]; }
        if (p >= prev_end) {
            const long long q = p + shift;
            if (q < cap) out[q] = text[p]; else latch_status(d_status, ANON_ERR_CAPACITY);
        }
    }
}

__global__ void __launch_bounds__(256) splice_tokens_kernel(long long S, const long long* __restrict__ D,
                                                            const long long* __restrict__ astart, const uint8_t* __restrict__ tok,
                                                            const long long* __restrict__ tok_off, uint8_t* __restrict__ out,
                                                            long long cap, int* d_status)
{
    const long long s = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= S) return;
    const long long q = astart[s] + D[s], a = tok_off[s], n = tok_off[s + 1] - a;
    if (q + n > cap) { latch_status(d_status, ANON_ERR_CAPACITY); return; }
    for (long long j = 0; j < n; j++) out[q + j] = tok[a + j];
}

__global__ void __launch_bounds__(256) splice_record_offsets_kernel(const long long* __restrict__ rec_off, int R, const anon_span* __restrict__ spans,
                                                                    long long S, const long long* __restrict__ D, long long* __restrict__ new_off)
{
    const int r = blockIdx.x * blockDim.x + threadIdx.x;
    if (r > R) return;
    long long lo = 0, hi = S;                       // number of spans in records < r
    while (lo < hi) { const long long mid = (lo + hi) >> 1; if (spans[mid].record_id < r) lo = mid + 1; else hi = mid; }
    new_off[r] = rec_off[r] + D[lo];
}

}  // namespace

int splice_records_impl(anon_ctx* ctx, WsCursor& ws, const uint8_t* d_text, size_t text_bytes, const int64_t* d_rec_off, int32_t R,
                        const anon_span* d_spans, int32_t S, const uint8_t* d_tok, const int64_t* d_tok_off,
                        uint8_t* d_new_text, size_t cap, int64_t* d_new_rec_off)
{
    if (!ctx || R < 0 || S < 0 || !d_rec_off || !d_new_rec_off || (text_bytes > 0 && (!d_text || !d_new_text)) ||
        (S > 0 && (!d_spans || !d_tok_off)))
        return ANON_ERR_INVALID_ARG;
    cudaStream_t st = ctx->stream;
    long long* D = (long long*)ws.take(((size_t)S + 1) * 8);
    long long* astart = (long long*)ws.take(((size_t)S + 1) * 8);
    long long* aend = (long long*)ws.take(((size_t)S + 1) * 8);
    long long* agg = (long long*)ws.take(scan::agg_bytes<long long>(S > 0 ? S : 1));
    if (!D || !astart || !aend || !agg) return ANON_ERR_OOM;
    ProfScope ps(ctx, PROF_DECODE, (double)text_bytes * 2 + (double)S * 64, 6);
    if (S > 0) {
        DeltaIn din{d_spans, (const long long*)d_tok_off};
        scan::reduce_and_scan<long long, scan::SumI64>(din, S, nullptr, agg, st);
        scan::apply<long long, scan::SumI64>(din, DeltaOut{d_spans, (const long long*)d_rec_off, D, astart, aend, S}, S, nullptr, agg, st);
    } else {
        CU_TRY(ctx, cudaMemsetAsync(D, 0, 8, st));
    }
    if (text_bytes > 0) {
        const long long chunks = ((long long)text_bytes + 15) / 16;
        splice_copy_kernel<<<(unsigned)((chunks + 255) / 256), 256, 0, st>>>(d_text, (long long)text_bytes, S, D, astart, aend,
                                                                           d_new_text, (long long)cap, ctx->d_status);
    }
    if (S > 0)
        splice_tokens_kernel<<<(unsigned)((S + 255) / 256), 256, 0, st>>>(S, D, astart, d_tok, (const long long*)d_tok_off, d_new_text,
                                                                         (long long)cap, ctx->d_status);
    splice_record_offsets_kernel<<<(unsigned)((R + 1 + 255) / 256), 256, 0, st>>>((const long long*)d_rec_off, R, d_spans, S, D,
                                                                                 (long long*)d_new_rec_off);
    CU_LAUNCH_CHECK(ctx, "splice_records");
    return ANON_OK;
}

extern "C" int anon_splice_records(anon_ctx* ctx, const uint8_t* d_text, size_t text_bytes, const int64_t* d_record_offsets, int32_t R,
                                   const anon_span* d_spans, int32_t S, const uint8_t* d_out_tokens, const int64_t* d_out_offsets,
                                   uint8_t* d_new_text, size_t new_text_capacity, int64_t* d_new_record_offsets)
{
    if (!ctx) return ANON_ERR_INVALID_ARG;
    CU_TRY(ctx, cudaSetDevice(ctx->device));
    WsCursor ws = ws_begin(ctx);
    return splice_records_impl(ctx, ws, d_text, text_bytes, d_record_offsets, R, d_spans, S, d_out_tokens, d_out_offsets,
                               d_new_text, new_text_capacity, d_new_record_offsets);
}

int decode_spans_impl(anon_ctx* ctx, WsCursor& ws, const int32_t* d_labels, const anon_tok_meta* d_meta, int32_t T,
                      int32_t num_labels, anon_span* d_spans, int32_t cap, int32_t* d_num)
{
    if (!ctx || T < 0 || cap < 0 || !d_num || (T > 0 && (!d_labels || !d_meta)) || (cap > 0 && !d_spans))
        return ANON_ERR_INVALID_ARG;
    if (num_labels < 1 || (num_labels & 1) == 0) return ANON_ERR_UNSUPPORTED;
    cudaStream_t st = ctx->stream;
    if (T == 0) { CU_TRY(ctx, cudaMemsetAsync(d_num, 0, 4, st)); return ANON_OK; }
    int* prev = (int*)ws.take((size_t)T * 4);
    int* agg_i = (int*)ws.take(scan::agg_bytes<int>(T));
    long long* agg_l = (long long*)ws.take(scan::agg_bytes<long long>(T));
    if (!prev || !agg_i || !agg_l) return ANON_ERR_OOM;
    ProfScope ps(ctx, PROF_DECODE, (double)T * 20 + (double)T * 8, 7);
    KeepIn kin{d_meta};
    scan::reduce_and_scan<int, scan::MaxI32>(kin, T, nullptr, agg_i, st);
    scan::apply<int, scan::MaxI32>(kin, PrevKeptOut{prev}, T, nullptr, agg_i, st);
    StartIn sin{d_labels, d_meta, prev};
    scan::reduce_and_scan<long long, scan::SumI64>(sin, T, nullptr, agg_l, st);
    scan::apply<long long, scan::SumI64>(sin, StartOut{d_labels, d_meta, prev, d_spans, cap}, T, nullptr, agg_l, st);
    decode_finish_kernel<<<1, 1, 0, st>>>(d_labels, d_meta, prev, T, agg_l + scan::num_tiles(T), d_spans, cap, d_num,
                                          ctx->d_status);
    CU_LAUNCH_CHECK(ctx, "decode_spans");
    return ANON_OK;
}

int gather_spans_impl(anon_ctx* ctx, WsCursor& ws, const uint8_t* d_text, const int64_t* d_rec_off,
                      const anon_span* d_spans, const int32_t* d_num_spans, int32_t S_max,
                      uint8_t* d_bytes, size_t cap, int64_t* d_off, uint8_t* d_type)
{
    if (!ctx || S_max < 0 || !d_off || (S_max > 0 && (!d_text || !d_rec_off || !d_spans))) return ANON_ERR_INVALID_ARG;
    cudaStream_t st = ctx->stream;
    if (S_max == 0) { CU_TRY(ctx, cudaMemsetAsync(d_off, 0, 8, st)); return ANON_OK; }
    long long* agg = (long long*)ws.take(scan::agg_bytes<long long>(S_max));
    if (!agg) return ANON_ERR_OOM;
    ProfScope ps(ctx, PROF_DECODE, (double)S_max * 40, 4);
    LenIn lin{d_spans};
    scan::reduce_and_scan<long long, scan::SumI64>(lin, S_max, d_num_spans, agg, st);
    scan::apply<long long, scan::SumI64>(lin, GatherOut{d_spans, d_text, (const long long*)d_rec_off, d_bytes,
                                                         (long long)cap, (long long*)d_off, d_type, ctx->d_status},
                                         S_max, d_num_spans, agg, st);
    gather_finish_kernel<<<1, 1, 0, st>>>(agg + scan::num_tiles(S_max), d_num_spans, S_max, (long long*)d_off);
    CU_LAUNCH_CHECK(ctx, "gather_spans");
    return ANON_OK;
}

extern "C" int anon_decode_spans(anon_ctx* ctx, const int32_t* d_labels, const anon_tok_meta* d_meta, int32_t T,
                                 int32_t num_labels, anon_span* d_spans, int32_t span_capacity, int32_t* d_num_spans)
{
    if (!ctx) return ANON_ERR_INVALID_ARG;
    CU_TRY(ctx, cudaSetDevice(ctx->device));
    WsCursor ws = ws_begin(ctx);
    return decode_spans_impl(ctx, ws, d_labels, d_meta, T, num_labels, d_spans, span_capacity, d_num_spans);
}

extern "C" int anon_gather_spans(anon_ctx* ctx, const uint8_t* d_text, const int64_t* d_record_offsets,
                                 const anon_span* d_spans, int32_t S, uint8_t* d_span_bytes, size_t bytes_capacity,
                                 int64_t* d_span_offsets, uint8_t* d_span_type)
{
    if (!ctx) return ANON_ERR_INVALID_ARG;
    CU_TRY(ctx, cudaSetDevice(ctx->device));
    WsCursor ws = ws_begin(ctx);
    return gather_spans_impl(ctx, ws, d_text, d_record_offsets, d_spans, nullptr, S, d_span_bytes, bytes_capacity,
                             d_span_offsets, d_span_type);
}
