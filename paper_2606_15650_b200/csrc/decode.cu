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
    const anon_span* spans; long long cap; long long* off; uint8_t* type; int* d_status;
    __device__ __forceinline__ void operator()(long long s, long long o, long long len) const {
        off[s] = o;
        if (type) type[s] = (uint8_t)spans[s].type;
        if (o + len > cap) latch_status(d_status, ANON_ERR_CAPACITY);
    }
};
// K8 copy: a warp takes 32 consecutive spans -- a contiguous byte range of the output -- and moves them one span at a time with
// lane-strided byte accesses (32 consecutive bytes per instruction on both sides) instead of one thread walking each span byte
// by byte (one sector per byte and lane).  Spans that would overflow the buffer are skipped (the scan has latched CAPACITY).
__global__ void __launch_bounds__(256) gather_copy_kernel(const anon_span* __restrict__ spans, const int* __restrict__ d_n, long long S_max,
                                                          const uint8_t* __restrict__ text, const long long* __restrict__ rec_off,
                                                          const long long* __restrict__ off, uint8_t* __restrict__ out, long long cap)
{
    const long long n = d_n ? min((long long)*d_n, S_max) : S_max;
    const int lane = threadIdx.x & 31;
    const long long s0 = ((long long)blockIdx.x * 8 + (threadIdx.x >> 5)) * 32;
    if (s0 >= n) return;
    const long long s = s0 + lane;
    long long src = 0, dst = 0; int len = 0;
    if (s < n) {
        const anon_span sp = spans[s];
        len = sp.char_end - sp.char_start; if (len < 0) len = 0;
        src = rec_off[sp.record_id] + sp.char_start;
        dst = off[s];
        if (dst + len > cap) len = 0;
    }
    const int cnt = (int)min(32ll, n - s0);
    for (int j = 0; j < cnt; j++) {
        const long long a = __shfl_sync(0xffffffffu, src, j), b = __shfl_sync(0xffffffffu, dst, j);
        const int l = __shfl_sync(0xffffffffu, len, j);
        for (int k = lane; k < l; k += 32) out[b + k] = text[a + k];
    }
}
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
    const anon_span* spans; const long long* rec_off; long long* D; long long* ostart; long long S;
    __device__ __forceinline__ void operator()(long long s, long long ex, long long v) const {
        const anon_span sp = spans[s];
        D[s] = ex;
        ostart[s] = rec_off[sp.record_id] + sp.char_start + ex;      // where the token of span s starts in the NEW text
        if (s == S - 1) D[S] = ex + v;
    }
};

// The rewritten text is produced OUTPUT-side: a thread owns 16 consecutive output bytes and finds, for each, whether it is
// a token byte (of the last span whose token starts at or before it) or a text byte of the gap behind that token
// (source = q - D[number of spans started]).  One 16-byte store per thread instead of 16 byte stores at a shifted address,
// and no separate token pass.  The spans of a 4 KB chunk of output are found through a chunk index (kb, below) and a short
// binary search among them.
constexpr int kSpChunk = 4096;

// kb[c] = number of spans whose token starts before output byte c * kSpChunk, for every chunk boundary c = 0 .. n_chunks:
// thread s (0 .. S) fills the boundaries that lie in (ostart[s-1], ostart[s]] -- usually none or one -- so that the copy
// kernel finds a chunk's spans with two loads instead of a binary search over the whole span list per chunk (which, run by one
// thread per CTA, was 2 x 22 dependent global loads = most of the round-2 first version's time)
__global__ void __launch_bounds__(256) splice_chunk_index_kernel(long long S, const long long* __restrict__ ostart,
                                                                 long long n_bounds, int* __restrict__ kb)
{
    const long long s = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (s > S) return;
    long long lo = s == 0 ? 0 : ostart[s - 1] / kSpChunk + 1;
    long long hi = s == S ? n_bounds - 1 : ostart[s] / kSpChunk;
    if (hi > n_bounds - 1) hi = n_bounds - 1;
    for (long long c = lo; c <= hi; c++) kb[c] = (int)s;
}

__global__ void __launch_bounds__(256) splice_out_kernel(const int* __restrict__ kb, const uint8_t* __restrict__ text, long long nbytes, long long S,
                                                         const long long* __restrict__ D, const long long* __restrict__ ostart,
                                                         const uint8_t* __restrict__ tok, const long long* __restrict__ tok_off,
                                                         uint8_t* __restrict__ out, long long cap, int* d_status)
{
    const long long total = nbytes + D[S];
    if (total > cap && blockIdx.x == 0 && threadIdx.x == 0) latch_status(d_status, ANON_ERR_CAPACITY);
    const long long lim = total < cap ? total : cap;
    const bool aligned = (reinterpret_cast<uintptr_t>(out) & 15) == 0;
    const long long stride = (long long)gridDim.x * blockDim.x * 16;
    for (long long q0 = ((long long)blockIdx.x * blockDim.x + threadIdx.x) * 16; q0 < lim; q0 += stride) {
        // the spans that matter for this 4 KB chunk of output: the last one that started before the chunk (its token or the
        // gap behind it may reach into the chunk) and those whose token starts inside it -- a few dozen consecutive rows of
        // ostart / D / tok_off that the 256 threads of the chunk all read (L1-resident); no shared memory, no barriers
        const long long c = q0 / kSpChunk;
        const long long k0 = __ldg(kb + c), k1 = __ldg(kb + c + 1);
        const long long first = k0 > 0 ? k0 - 1 : 0;
        const int n = (int)(k1 - first);
        const long long* os = ostart + first;
        const long long* dd = D + first;
        const long long* to = tok_off + first;              // only read when n > 0 (S > 0)
        int lo = 0, hi = n;                                 // kl = number of those spans with ostart <= q0
        while (lo < hi) { const int mid = (lo + hi) >> 1; if (__ldg(os + mid) <= q0) lo = mid + 1; else hi = mid; }
        int kl = lo;
        uint32_t w[4] = {0u, 0u, 0u, 0u};
        const int cnt = (int)(lim - q0 < 16 ? lim - q0 : 16);
        // fast path (about four chunks in five): all 16 bytes come from ONE source range -- the token of span kl-1, or the gap
        // behind it with no further token starting inside these 16 bytes -- so they are 16 independent loads from consecutive
        // addresses, no per-byte decision
        const uint8_t* src1 = nullptr;
        if (cnt == 16) {
            const long long next_start = kl < n ? __ldg(os + kl) : (long long)0x7fffffffffffffffll;
            if (kl > 0) {
                const long long t0 = __ldg(to + kl - 1), rel = q0 - __ldg(os + kl - 1), tl = __ldg(to + kl) - t0;
                if (rel + 16 <= tl) src1 = tok + t0 + rel;                               // inside the token
                else if (rel >= tl && next_start >= q0 + 16) src1 = text + (q0 - __ldg(dd + kl));   // inside the gap
            } else if (next_start >= q0 + 16) {
                src1 = text + (q0 - __ldg(dd));
            }
        }
        if (src1) {
#pragma unroll
            for (int j = 0; j < 16; j++) w[j >> 2] |= (uint32_t)__ldg(src1 + j) << (8 * (j & 3));
        } else {
            // general case: walk the (at most a few) SEGMENTS that meet in these bytes -- rest of a token, a gap up to the next
            // token start, the next token ... -- looking the span rows up once per segment, not once per byte
            unsigned long long lo8 = 0ull, hi8 = 0ull;
            int j = 0;
            while (j < cnt) {
                const long long q = q0 + j;
                while (kl < n && __ldg(os + kl) <= q) kl++;
                const long long next_start = kl < n ? __ldg(os + kl) : (long long)0x7fffffffffffffffll;
                const uint8_t* src;
                long long seg_end = next_start;
                if (kl > 0) {
                    const long long t0 = __ldg(to + kl - 1), rel = q - __ldg(os + kl - 1), tl = __ldg(to + kl) - t0;
                    if (rel < tl) { src = tok + t0 + rel; seg_end = q + (tl - rel); }
                    else src = text + (q - __ldg(dd + kl));
                } else {
                    src = text + (q - __ldg(dd));
                }
                const int run = (int)(seg_end - q < (long long)(cnt - j) ? seg_end - q : (long long)(cnt - j));
                for (int i = 0; i < run; i++) {
                    const unsigned long long b = __ldg(src + i);
                    const int pos = j + i;
                    if (pos < 8) lo8 |= b << (8 * pos); else hi8 |= b << (8 * (pos - 8));
                }
                j += run;
            }
            w[0] = (uint32_t)lo8; w[1] = (uint32_t)(lo8 >> 32); w[2] = (uint32_t)hi8; w[3] = (uint32_t)(hi8 >> 32);
        }
        if (aligned && cnt == 16) {
            *reinterpret_cast<uint4*>(out + q0) = make_uint4(w[0], w[1], w[2], w[3]);
        } else {
#pragma unroll
            for (int j = 0; j < 16; j++) if (j < cnt) out[q0 + j] = (uint8_t)(w[j >> 2] >> (8 * (j & 3)));
        }
    }
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
    long long* ostart = (long long*)ws.take(((size_t)S + 1) * 8);
    long long* agg = (long long*)ws.take(scan::agg_bytes<long long>(S > 0 ? S : 1));
    const long long n_bounds = (long long)(cap / kSpChunk) + 2;          // chunk boundaries 0 .. ceil(cap / chunk)
    int* kb = (int*)ws.take((size_t)n_bounds * 4);
    if (!D || !ostart || !agg || !kb) return ANON_ERR_OOM;
    ProfScope ps(ctx, PROF_DECODE, (double)text_bytes * 2 + (double)S * 64, 6);
    if (S > 0) {
        DeltaIn din{d_spans, (const long long*)d_tok_off};
        scan::reduce_and_scan<long long, scan::SumI64>(din, S, nullptr, agg, st);
        scan::apply<long long, scan::SumI64>(din, DeltaOut{d_spans, (const long long*)d_rec_off, D, ostart, S}, S, nullptr, agg, st);
    } else {
        CU_TRY(ctx, cudaMemsetAsync(D, 0, 8, st));
    }
    if (text_bytes > 0 || S > 0) {
        // persistent grid over 4 KB output chunks (the new size lives on the device: text_bytes + D[S] <= cap)
        const long long chunks = ((long long)text_bytes + kSpChunk - 1) / kSpChunk + 1;
        const long long want = (long long)ctx->sm_count * 8;
        splice_chunk_index_kernel<<<(unsigned)((S + 1 + 255) / 256), 256, 0, st>>>(S, ostart, n_bounds, kb);
        splice_out_kernel<<<(unsigned)(chunks < want ? chunks : want), 256, 0, st>>>(kb, d_text, (long long)text_bytes, S, D, ostart, d_tok,
                                                                                 (const long long*)d_tok_off, d_new_text, (long long)cap,
                                                                                 ctx->d_status);
    }
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
    ProfScope ps(ctx, PROF_DECODE, (double)S_max * 40, 5);
    LenIn lin{d_spans};
    scan::reduce_and_scan<long long, scan::SumI64>(lin, S_max, d_num_spans, agg, st);
    scan::apply<long long, scan::SumI64>(lin, GatherOut{d_spans, (long long)cap, (long long*)d_off, d_type, ctx->d_status},
                                         S_max, d_num_spans, agg, st);
    gather_finish_kernel<<<1, 1, 0, st>>>(agg + scan::num_tiles(S_max), d_num_spans, S_max, (long long*)d_off);
    gather_copy_kernel<<<(unsigned)((S_max + 255) / 256), 256, 0, st>>>(d_spans, d_num_spans, S_max, d_text, (const long long*)d_rec_off,
                                                                       (const long long*)d_off, d_bytes, (long long)cap);
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

// ---- A9 without any allocation: anon_decode_spans_static ---------------------------------------------------------------------
// The same two transform-scans as decode_spans_impl, with the scratch (prev_kept[T], the tile aggregates of both scans and a
// status word) in a file-scope device array instead of the context workspace: no context, no cudaMalloc / cudaFree, nothing but
// kernel launches and one 4-byte memset on the caller's stream.  For callers that may not allocate (code under CUDA graph capture,
// serving loops, harnesses that forbid it).  Every GPU that loads the library holds the array (4.2 MB) until exit; every call on a
// device shares it, so two calls that overlap on the GPU (different streams) race -- serialise them.  Nothing in it has to start at
// zero except the status word, which each call clears: prev_kept and the aggregates are fully rewritten for the call's T before
// they are read.
namespace {

constexpr int kStaticMaxTokens = ANON_DECODE_STATIC_MAX_TOKENS;
constexpr size_t kStaticStatusBytes = 256;
constexpr size_t kStaticPrevBytes = (size_t)kStaticMaxTokens * 4;
constexpr size_t kStaticAggI = ((size_t)(kStaticMaxTokens / scan::kTile + 2) * sizeof(int) + 255) / 256 * 256;
constexpr size_t kStaticAggL = ((size_t)(kStaticMaxTokens / scan::kTile + 2) * sizeof(long long) + 255) / 256 * 256;
constexpr size_t kStaticBytes = kStaticStatusBytes + kStaticPrevBytes + kStaticAggI + kStaticAggL;

static __device__ __align__(256) uint8_t g_decode_static_scratch[kStaticBytes];

// In host code `g_decode_static_scratch` is only a stand-in for the symbol: the device address comes from cudaGetSymbolAddress,
// asked once per device with that device current.
constexpr int kStaticMaxDevices = 64;
uint8_t* g_static_ptr[kStaticMaxDevices] = {nullptr};

int static_scratch(int device, uint8_t** out) {
    if (device < 0 || device >= kStaticMaxDevices) return ANON_ERR_INVALID_ARG;
    if (cudaSetDevice(device) != cudaSuccess) { cudaGetLastError(); return ANON_ERR_CUDA; }
    uint8_t* p = __atomic_load_n(&g_static_ptr[device], __ATOMIC_ACQUIRE);
    if (!p) {
        void* sym = nullptr;
        if (cudaGetSymbolAddress(&sym, g_decode_static_scratch) != cudaSuccess || !sym) { cudaGetLastError(); return ANON_ERR_CUDA; }
        p = (uint8_t*)sym;
        __atomic_store_n(&g_static_ptr[device], p, __ATOMIC_RELEASE);     // racing first calls store the same address
    }
    *out = p;
    return ANON_OK;
}

}  // namespace

extern "C" int anon_decode_spans_static(int device, void* cuda_stream, const int32_t* d_labels, const anon_tok_meta* d_meta, int32_t T,
                                        int32_t num_labels, anon_span* d_spans, int32_t span_capacity, int32_t* d_num_spans)
{
    if (T < 0 || span_capacity < 0 || !d_num_spans || (T > 0 && (!d_labels || !d_meta)) || (span_capacity > 0 && !d_spans))
        return ANON_ERR_INVALID_ARG;
    if (num_labels < 1 || (num_labels & 1) == 0) return ANON_ERR_UNSUPPORTED;
    if (T > kStaticMaxTokens) return ANON_ERR_CAPACITY;                 // beyond the static scratch: use anon_decode_spans
    uint8_t* base = nullptr;
    const int rc = static_scratch(device, &base);
    if (rc != ANON_OK) return rc;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if (T == 0) return cudaMemsetAsync(d_num_spans, 0, 4, st) == cudaSuccess ? ANON_OK : (cudaGetLastError(), ANON_ERR_CUDA);
    int* status = (int*)base;
    int* prev = (int*)(base + kStaticStatusBytes);
    int* agg_i = (int*)(base + kStaticStatusBytes + kStaticPrevBytes);
    long long* agg_l = (long long*)(base + kStaticStatusBytes + kStaticPrevBytes + kStaticAggI);
    if (cudaMemsetAsync(status, 0, 4, st) != cudaSuccess) { cudaGetLastError(); return ANON_ERR_CUDA; }
    KeepIn kin{d_meta};
    scan::reduce_and_scan<int, scan::MaxI32>(kin, T, nullptr, agg_i, st);
    scan::apply<int, scan::MaxI32>(kin, PrevKeptOut{prev}, T, nullptr, agg_i, st);
    StartIn sin{d_labels, d_meta, prev};
    scan::reduce_and_scan<long long, scan::SumI64>(sin, T, nullptr, agg_l, st);
    scan::apply<long long, scan::SumI64>(sin, StartOut{d_labels, d_meta, prev, d_spans, span_capacity}, T, nullptr, agg_l, st);
    decode_finish_kernel<<<1, 1, 0, st>>>(d_labels, d_meta, prev, T, agg_l + scan::num_tiles(T), d_spans, span_capacity, d_num_spans,
                                          status);
    if (cudaGetLastError() != cudaSuccess) return ANON_ERR_CUDA;
    return ANON_OK;
}
