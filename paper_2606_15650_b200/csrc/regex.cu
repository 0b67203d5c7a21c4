// regex.cu -- NEXT-4: the regex detector as a table-driven DFA scan, and the regex / NER span merge.
// P:L43 ("21 custom regex patterns" beside the transformer NER), P:L170 (overlap resolution); S8f NEXT-4; rules D17-D19 of
// DESIGN.md.  Integer / byte work: bit-exact against oracle/regex_layer.py.
//
// The automaton comes from the host compiler (regex_dfa.py): one DFA for all patterns, over byte classes, anchored at the
// candidate start.  Rule D18 (leftmost-longest, non-overlapping, word boundaries, lowest pattern index) in three passes:
//   R1  regex_candidates_kernel   every byte position in parallel: the longest match that starts there (0 = none).  Tables
//                                 and a text tile (+ max_match look-ahead) live in shared memory; most positions die on
//                                 their first transition.  Writes one u16 per byte: len | pattern << 8.
//   R2  regex_select_kernel       one warp per record walks the candidates left to right, 128 positions per step, from
//                                 2048-position chunks staged in shared memory: the first candidate at or after the cursor
//                                 is selected (bit 15), the cursor jumps to its end.
//   R3  scan of the per-record counts, then regex_write_kernel compacts the selected candidates into the span list in
//       stream order (ballot + popc ranks inside a warp).
// Merge (D19): per NER span one binary search in the regex list (sorted, non-overlapping) decides keep / drop; a scan of
// the keep flags plus cross ranks (binary searches) gives every surviving span its slot in the merged list.
#include "common.cuh"
#include "scan.cuh"

#include <new>

struct anon_regex {
    anon_ctx* ctx = nullptr;
    uint8_t* d_tab = nullptr;        // cw[256], type_of[256], tr[n_states * n_classes] (see regex_candidates_kernel)
    uint32_t tab_bytes = 0;          // padded to 16 bytes
    uint32_t smem_bytes = 0;         // dynamic shared memory of regex_candidates_kernel
    int ctas_per_sm = 1;             // resident CTAs of regex_candidates_kernel per SM (sizes its persistent grid)
    int n_states = 0, n_classes = 0, n_patterns = 0, max_match = 0;
};

namespace {

constexpr uint32_t kMagic = 0x31585241u;     // 'ARX1'
constexpr int kTile = 4096;                  // byte positions per tile of R1
constexpr int kThreads = 256;
constexpr int kTextSmem = kTile + 256 + 48;  // tile + look-ahead (max_match <= 255) + alignment slack
constexpr int kStartWords = (kTile + 256) / 32 + 1;
constexpr int kShortWalk = 8;                // steps of the first walking pass of R1

// largest r in [lo, hi] with off[r] <= p  (off[lo] <= p is given)
__device__ __forceinline__ int record_of(const long long* __restrict__ off, int lo, int hi, long long p) {
    while (lo < hi) {
        const int mid = (lo + hi + 1) >> 1;
        if (off[mid] <= p) lo = mid; else hi = mid - 1;
    }
    return lo;
}

// tile_rec[t] = record that holds the first byte of tile t (t = 0 .. n_tiles; the last entry closes the last tile)
__global__ void __launch_bounds__(kThreads) regex_tile_records_kernel(const long long* __restrict__ rec_off, int R, long long nbytes,
                                                                      long long n_tiles, int* __restrict__ tile_rec)
{
    const long long t = (long long)blockIdx.x * kThreads + threadIdx.x;
    if (t > n_tiles) return;
    const long long p = t * kTile < nbytes ? t * kTile : nbytes - 1;
    tile_rec[t] = record_of(rec_off, 0, R - 1, p);
}

__device__ __forceinline__ uint32_t lds_u8(uint32_t addr) { uint32_t v; asm volatile("ld.shared.u8 %0, [%1];" : "=r"(v) : "r"(addr)); return v; }
__device__ __forceinline__ uint32_t lds_u32(uint32_t addr) { uint32_t v; asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(addr)); return v; }

// One DFA walk from a start position: the longest accepting prefix that ends on a word boundary, as len | pattern << 8.
// `left` = bytes to the end of the record (capped), `lim` = steps allowed in this call.  Returns true if the automaton is
// still alive after `lim` steps (the caller may walk on with a larger `lim`).  All operands are 32-bit shared-memory
// addresses (text byte, cw table, transition table): ~14 instructions and one dependent load per step.
__device__ __forceinline__ bool dfa_walk(uint32_t b, int left, int lim, uint32_t cw, uint32_t tr, int n_classes, uint32_t& out)
{
    uint32_t st = 1, cwn = lds_u8(cw + lds_u8(b));
    out = 0;
    int i = 0;
    while (i < lim) {
        const uint32_t cwi = cwn;
        cwn = lds_u8(cw + lds_u8(b + i + 1));                                   // inside the staged look-ahead for every i < lim
        if (i + 1 >= left) cwn = 0u;                                            // the record's edge counts as a non-word byte
        const uint32_t t = lds_u32(tr + ((st * n_classes + (cwi & 0x7f)) << 2));
        st = t & 0xffffu;
        if (st == 0) return false;
        ++i;
        if ((t >> 16) && !(cwn & 0x80)) out = (uint32_t)i | (((t >> 16) - 1) << 8);
    }
    return true;
}

// Device tables (built by anon_regex_load): cw[256] = class | is_word << 7, type_of[256], then tr[state * n_classes + class] =
// next state | (accept(next state) + 1) << 16 -- one dependent shared-memory load per DFA step.
__global__ void __launch_bounds__(kThreads) regex_candidates_kernel(
    const uint8_t* __restrict__ tab, uint32_t tab_bytes, int n_classes, int max_match,
    const uint8_t* __restrict__ text, long long nbytes, const long long* __restrict__ rec_off, int R, const int* __restrict__ tile_rec,
    long long n_tiles, uint16_t* __restrict__ cand)
{
    extern __shared__ __align__(16) uint8_t smem[];
    uint8_t* s_tab = smem;
    uint8_t* s_text = smem + tab_bytes;
    uint16_t* s_cand = reinterpret_cast<uint16_t*>(s_text + kTextSmem);     // longest match per position of the tile
    uint16_t* s_list = s_cand + kTile;                                      // positions that start a walk
    uint16_t* s_surv = s_list + kTile;                                      // starts whose walk outlives the short first pass
    __shared__ uint32_t s_recbits[kStartWords];                             // record starts inside the tile and its look-ahead
    __shared__ uint32_t s_startbits[kTile / 32];                            // positions that can start a match
    __shared__ int s_wtot[kThreads / 32];
    __shared__ int s_nsurv;
    for (uint32_t i = threadIdx.x; i < tab_bytes / 16; i += kThreads)
        reinterpret_cast<uint4*>(s_tab)[i] = reinterpret_cast<const uint4*>(tab)[i];
    const uint8_t* cw = s_tab;
    const uint32_t* tr = reinterpret_cast<const uint32_t*>(s_tab + 512);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;

    for (long long tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
        const long long tile0 = tile * kTile;
        const long long lo = tile0 > 0 ? tile0 - 1 : 0;
        long long hi = tile0 + kTile + max_match;
        if (hi > nbytes) hi = nbytes;
        // stage text[lo, hi) through aligned 16-byte loads (a chunk that holds one valid byte is readable as a whole)
        const uintptr_t g0 = reinterpret_cast<uintptr_t>(text + lo) & ~(uintptr_t)15;
        const int nchunk = (int)((reinterpret_cast<uintptr_t>(text + hi) - g0 + 15) >> 4);
        __syncthreads();                               // previous tile fully consumed (and s_tab written, first time)
        for (int i = threadIdx.x; i < nchunk; i += kThreads)
            reinterpret_cast<uint4*>(s_text)[i] = __ldg(reinterpret_cast<const uint4*>(g0) + i);
        for (int i = threadIdx.x; i < kTile / 8; i += kThreads) reinterpret_cast<uint4*>(s_cand)[i] = make_uint4(0, 0, 0, 0);
        if (threadIdx.x < kStartWords) s_recbits[threadIdx.x] = 0;
        if (threadIdx.x == 0) s_nsurv = 0;
        __syncthreads();
        // record starts (and the end of the text, rec_off[R]) in [tile0, tile0 + kTile + 256): the left word boundary of rule D18
        // and the distance from a start position to the end of its record both come from these bits
        for (int r = tile_rec[tile] + threadIdx.x; r <= R; r += kThreads) {
            const long long o = rec_off[r] - tile0;
            if (o >= kTile + 256) break;
            if (o >= 0) atomicOr(&s_recbits[o >> 5], 1u << (o & 31));
        }
        __syncthreads();
        const uint8_t* tbase = s_text + ((long long)(reinterpret_cast<uintptr_t>(text) - g0) + tile0);   // tile position 0
        const int n_here = (int)(nbytes - tile0 < kTile ? nbytes - tile0 : kTile);
        const uint32_t tbase_s = (uint32_t)__cvta_generic_to_shared(tbase);
        const uint32_t cw_s = (uint32_t)__cvta_generic_to_shared(cw), tr_s = (uint32_t)__cvta_generic_to_shared(tr);
        // A: which positions can start a match (first transition alive, word boundary on the left)?  Four per thread.
#pragma unroll
        for (int k = 0; k < kTile / 4 / kThreads; k++) {
            const int q = k * kThreads + threadIdx.x, o = q * 4;
            uint32_t nib = 0;
            if (o < n_here) {
                const uint32_t rb = (s_recbits[q >> 3] >> ((q & 7) * 4)) & 0xfu;
                uint32_t prev_word = (o > 0 || tile0 > 0) ? (cw[tbase[o - 1]] & 0x80u) : 0u;
#pragma unroll
                for (int j = 0; j < 4; j++) {
                    const uint32_t c = cw[tbase[o + j]];
                    const bool alive = (tr[n_classes + (c & 0x7f)] & 0xffffu) != 0;
                    if (alive && o + j < n_here && (!prev_word || ((rb >> j) & 1u))) nib |= 1u << j;
                    prev_word = c & 0x80u;
                }
            }
            uint32_t v = nib << ((lane & 7) * 4);
            v |= __shfl_xor_sync(0xffffffffu, v, 1);
            v |= __shfl_xor_sync(0xffffffffu, v, 2);
            v |= __shfl_xor_sync(0xffffffffu, v, 4);
            if ((lane & 7) == 0) s_startbits[q >> 3] = v;
        }
        __syncthreads();
        // compaction of the start bits into a position list: warp w owns 16 words, lanes 0..15 one word each
        uint32_t word = lane < 16 ? s_startbits[warp * 16 + lane] : 0u;
        int incl = __popc(word);
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const int t = __shfl_up_sync(0xffffffffu, incl, d);
            if (lane >= d) incl += t;
        }
        if (lane == 31) s_wtot[warp] = incl;
        __syncthreads();
        int pos = incl - __popc(word), n = 0;
#pragma unroll
        for (int w = 0; w < kThreads / 32; w++) {
            if (w < warp) pos += s_wtot[w];
            n += s_wtot[w];
        }
        while (word) {
            s_list[pos++] = (uint16_t)((warp * 16 + lane) * 32 + __ffs(word) - 1);
            word &= word - 1;
        }
        __syncthreads();
        // B: the walks.  First pass: every start, at most kShortWalk steps (most die on the next separator); the few that
        // are still alive are walked to the end in a second pass, so a warp never waits 80 steps for one long entity per round.
        for (int idx = threadIdx.x; idx < n; idx += kThreads) {
            const int o = s_list[idx];
            int w = o >> 5;                            // bytes to the end of the record = distance to the next record start
            uint32_t bits = s_recbits[w] & ~((2u << (o & 31)) - 1u);
            const int w_last = (o + max_match) >> 5;
            while (!bits && w < w_last) bits = s_recbits[++w];
            const int left = bits ? (w << 5) + __ffs(bits) - 1 - o : max_match + 1;
            const int limit = left < max_match ? left : max_match;
            uint32_t out;
            const bool alive = dfa_walk(tbase_s + o, left, limit < kShortWalk ? limit : kShortWalk, cw_s, tr_s, n_classes, out);
            if (alive && limit > kShortWalk) s_surv[atomicAdd(&s_nsurv, 1)] = (uint16_t)o;
            else s_cand[o] = (uint16_t)out;
        }
        __syncthreads();
        const int nsurv = s_nsurv;
        for (int idx = threadIdx.x; idx < nsurv; idx += kThreads) {
            const int o = s_surv[idx];
            int w = o >> 5;
            uint32_t bits = s_recbits[w] & ~((2u << (o & 31)) - 1u);
            const int w_last = (o + max_match) >> 5;
            while (!bits && w < w_last) bits = s_recbits[++w];
            const int left = bits ? (w << 5) + __ffs(bits) - 1 - o : max_match + 1;
            uint32_t out;
            dfa_walk(tbase_s + o, left, left < max_match ? left : max_match, cw_s, tr_s, n_classes, out);
            s_cand[o] = (uint16_t)out;
        }
        __syncthreads();
        // coalesced store of the tile's candidates (cand is padded, so the ragged last tile stores whole 16-byte words)
        for (int q = threadIdx.x; q * 8 < n_here; q += kThreads)
            reinterpret_cast<uint4*>(cand + tile0)[q] = reinterpret_cast<const uint4*>(s_cand)[q];
    }
}

// One warp per record.  The record's candidate words are staged through shared memory in chunks of kSelChunk positions
// (coalesced 16-byte loads), so that the walk itself -- find the first candidate at or after the cursor, select it, jump to
// its end -- runs at shared-memory latency: a 64 KB record costs 32 global round trips instead of one per selected span.
constexpr int kSelWarps = 4;
constexpr int kSelChunk = 2048;

__global__ void __launch_bounds__(kSelWarps * 32) regex_select_kernel(uint16_t* __restrict__ cand, const long long* __restrict__ rec_off, int R,
                                                                      int* __restrict__ rec_count)
{
    __shared__ __align__(16) uint16_t s_c[kSelWarps][kSelChunk];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int r = blockIdx.x * kSelWarps + warp;
    if (r >= R) return;
    long long s = rec_off[r];
    const long long re = rec_off[r + 1];
    uint16_t* sc = s_c[warp];
    int count = 0;
    while (s < re) {
        const long long cbase = s & ~7LL;                                       // 16-byte aligned entry
        long long nent = ((re - cbase) + 7) & ~7LL;                            // cand is padded: whole 16-byte words may be read
        if (nent > kSelChunk) nent = kSelChunk;
        for (int i = lane; i * 8 < nent; i += 32)
            reinterpret_cast<uint4*>(sc)[i] = reinterpret_cast<const uint4*>(cand + cbase)[i];
        __syncwarp();
        const long long cend = cbase + nent < re ? cbase + nent : re;          // positions of this chunk that belong to the record
        while (s < cend) {
            const long long wb = s & ~3LL, idx = wb + lane * 4;
            uint32_t c[4] = {0u, 0u, 0u, 0u};
            if (idx < cend) {
                const uint2 v = *reinterpret_cast<const uint2*>(sc + (idx - cbase));
                c[0] = v.x & 0xffffu; c[1] = v.x >> 16; c[2] = v.y & 0xffffu; c[3] = v.y >> 16;
            }
            int first = -1;
#pragma unroll
            for (int j = 3; j >= 0; j--)
                if ((c[j] & 0xffu) && idx + j >= s && idx + j < cend) first = j;
            const uint32_t any = __ballot_sync(0xffffffffu, first >= 0);
            if (!any) { s = wb + 128 < cend ? wb + 128 : cend; continue; }
            const int f = __ffs(any) - 1;
            const int fj = __shfl_sync(0xffffffffu, first, f);
            const uint32_t cv = __shfl_sync(0xffffffffu, first >= 0 ? c[first] : 0u, f);
            const long long pos = wb + f * 4 + fj;
            if (lane == f) cand[pos] = (uint16_t)(cv | 0x8000u);
            count++;
            s = pos + (cv & 0xffu);
        }
        __syncwarp();                                                          // the chunk is consumed: it may be overwritten
    }
    if (lane == 0) rec_count[r] = count;
}

struct CountIn {
    const int* cnt;
    __device__ __forceinline__ long long operator()(long long r) const { return cnt[r]; }
};
struct BaseOut {
    long long* base;
    __device__ __forceinline__ void operator()(long long r, long long ex, long long) const { base[r] = ex; }
};

__global__ void __launch_bounds__(kThreads) regex_write_kernel(const uint16_t* __restrict__ cand, const long long* __restrict__ rec_off, int R,
                                                               const long long* __restrict__ rec_base, const uint8_t* __restrict__ type_of,
                                                               anon_span* __restrict__ spans, long long cap)
{
    const int r = blockIdx.x * (kThreads / 32) + (threadIdx.x >> 5), lane = threadIdx.x & 31;
    if (r >= R) return;
    const long long rs = rec_off[r], re = rec_off[r + 1];
    long long o = rec_base[r];
    for (long long wb0 = rs & ~3LL; wb0 < re; wb0 += 512) {                     // four independent window loads in flight
        uint2 v[4];
#pragma unroll
        for (int u = 0; u < 4; u++) {
            const long long idx = wb0 + u * 128 + lane * 4;
            v[u] = idx < re ? *reinterpret_cast<const uint2*>(cand + idx) : make_uint2(0u, 0u);
        }
#pragma unroll
        for (int u = 0; u < 4; u++) {
            const long long idx = wb0 + u * 128 + lane * 4;
            uint32_t c[4] = {v[u].x & 0xffffu, v[u].x >> 16, v[u].y & 0xffffu, v[u].y >> 16};
#pragma unroll
            for (int j = 0; j < 4; j++)
                if (idx + j < rs || idx + j >= re) c[j] = 0;
            int n = 0;
#pragma unroll
            for (int j = 0; j < 4; j++) n += (c[j] >> 15) & 1;
            int incl = n;
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) {
                const int t = __shfl_up_sync(0xffffffffu, incl, d);
                if (lane >= d) incl += t;
            }
            long long k = o + incl - n;
#pragma unroll
            for (int j = 0; j < 4; j++) {
                if (c[j] & 0x8000u) {
                    if (k < cap) {
                        const int cs = (int)(idx + j - rs);
                        spans[k] = anon_span{r, cs, cs + (int)(c[j] & 0xffu), (int)type_of[(c[j] >> 8) & 0x7fu]};
                    }
                    k++;
                }
            }
            o += __shfl_sync(0xffffffffu, incl, 31);
        }
    }
}

__global__ void regex_finish_kernel(const long long* total, long long cap, int* d_num, int* d_status) {
    const long long n = *total;
    *d_num = (int)(n > 0x7fffffffLL ? 0x7fffffffLL : n);
    if (n > cap) latch_status(d_status, ANON_ERR_CAPACITY);
}

// ---- merge (D19) ----
__device__ __forceinline__ int dev_count(const int* d_n, int n_max) {
    if (!d_n) return n_max;
    const int n = *d_n;
    return n < 0 ? 0 : (n < n_max ? n : n_max);
}

__global__ void __launch_bounds__(kThreads) merge_flag_kernel(const anon_span* __restrict__ ner, const int* d_n_ner, int ner_max,
                                                              const anon_span* __restrict__ rgx, const int* d_n_rgx, int rgx_max,
                                                              uint8_t* __restrict__ keep, int* __restrict__ rgx_before)
{
    const int i = blockIdx.x * kThreads + threadIdx.x;
    const int n1 = dev_count(d_n_ner, ner_max), n2 = dev_count(d_n_rgx, rgx_max);
    if (i >= n1) return;
    const anon_span sp = ner[i];
    // first regex span that ends after sp starts: (record, char_end) > (sp.record, sp.char_start)
    int lo = 0, hi = n2;
    while (lo < hi) {
        const int mid = (lo + hi) >> 1;
        const anon_span q = rgx[mid];
        if (q.record_id < sp.record_id || (q.record_id == sp.record_id && q.char_end <= sp.char_start)) lo = mid + 1; else hi = mid;
    }
    const bool clash = lo < n2 && rgx[lo].record_id == sp.record_id && rgx[lo].char_start < sp.char_end;
    keep[i] = clash ? 0 : 1;
    // regex spans ordered strictly before sp: (record, char_start) < (sp.record, sp.char_start)
    int a = 0, b = n2;
    while (a < b) {
        const int mid = (a + b) >> 1;
        const anon_span q = rgx[mid];
        if (q.record_id < sp.record_id || (q.record_id == sp.record_id && q.char_start < sp.char_start)) a = mid + 1; else b = mid;
    }
    rgx_before[i] = a;
}

struct KeepIn {
    const uint8_t* keep;
    __device__ __forceinline__ long long operator()(long long i) const { return keep[i]; }
};
struct KeepOut {
    long long* kpos;
    __device__ __forceinline__ void operator()(long long i, long long ex, long long) const { kpos[i] = ex; }
};

__global__ void __launch_bounds__(kThreads) merge_write_kernel(const anon_span* __restrict__ ner, const int* d_n_ner, int ner_max,
                                                               const anon_span* __restrict__ rgx, const int* d_n_rgx, int rgx_max,
                                                               const uint8_t* __restrict__ keep, const int* __restrict__ rgx_before,
                                                               const long long* __restrict__ kpos, const long long* __restrict__ kept_total,
                                                               anon_span* __restrict__ out, long long cap, int* d_num, int* d_status)
{
    const long long i = (long long)blockIdx.x * kThreads + threadIdx.x;
    const int n1 = dev_count(d_n_ner, ner_max), n2 = dev_count(d_n_rgx, rgx_max);
    const long long kept = n1 > 0 ? *kept_total : 0;
    if (i == 0) {
        *d_num = (int)(kept + n2);
        if (kept + n2 > cap) latch_status(d_status, ANON_ERR_CAPACITY);
    }
    if (i < ner_max) {
        if (i < n1 && keep[i]) {
            const long long k = kpos[i] + rgx_before[i];
            if (k < cap) out[k] = ner[i];
        }
        return;
    }
    const long long j = i - ner_max;
    if (j >= n2) return;
    const anon_span q = rgx[j];
    int lo = 0, hi = n1;                                // NER spans ordered at or before q (ties: NER first)
    while (lo < hi) {
        const int mid = (lo + hi) >> 1;
        const anon_span sp = ner[mid];
        if (sp.record_id < q.record_id || (sp.record_id == q.record_id && sp.char_start <= q.char_start)) lo = mid + 1; else hi = mid;
    }
    const long long k = j + (lo < n1 ? kpos[lo] : kept);
    if (k < cap) out[k] = q;
}

}  // namespace

extern "C" int anon_regex_load(anon_ctx* ctx, const void* h_blob, size_t blob_bytes, anon_regex** out) {
    if (!ctx || !h_blob || !out) return ANON_ERR_INVALID_ARG;
    *out = nullptr;
    if (blob_bytes < 32 + 768) return ANON_ERR_INVALID_ARG;
    uint32_t head[8];
    memcpy(head, h_blob, 32);
    const uint64_t ns = head[1], nc = head[2], np = head[3], mm = head[4];
    if (head[0] != kMagic || ns < 2 || ns > 65535 || nc < 1 || nc > 256 || np < 1 || np > 127 || mm < 1 || mm > 255)
        return ANON_ERR_INVALID_ARG;
    const uint64_t off_accept = 768, off_trans = off_accept + (2 * ns + 3) / 4 * 4;
    if (blob_bytes != 32 + off_trans + 2 * ns * nc) return ANON_ERR_INVALID_ARG;
    const uint8_t* tab = (const uint8_t*)h_blob + 32;
    const int16_t* accept = (const int16_t*)(tab + off_accept);
    const uint16_t* trans = (const uint16_t*)(tab + off_trans);
    for (uint64_t c = 0; c < 256; c++) if (tab[c] >= nc) return ANON_ERR_INVALID_ARG;
    for (uint64_t s = 0; s < ns; s++) if (accept[s] < -1 || accept[s] >= (int)np) return ANON_ERR_INVALID_ARG;
    for (uint64_t i = 0; i < ns * nc; i++) if (trans[i] >= ns || (i < nc && trans[i] != 0)) return ANON_ERR_INVALID_ARG;
    if (accept[0] >= 0 || accept[1] >= 0) return ANON_ERR_INVALID_ARG;        // dead state / empty match
    if (nc > 128) return ANON_ERR_UNSUPPORTED;                                 // the class shares a byte with the word flag
    const uint64_t padded = (512 + 4 * ns * nc + 15) / 16 * 16;
    const uint64_t smem_need = padded + kTextSmem + 3 * kTile * 2;
    if (smem_need > (uint64_t)ctx->smem_optin) return ANON_ERR_UNSUPPORTED;    // tables must fit shared memory beside a tile
    std::vector<uint8_t> dev_tab(padded, 0);
    for (int c = 0; c < 256; c++) {
        dev_tab[c] = (uint8_t)(tab[c] | (tab[256 + c] ? 0x80 : 0));
        dev_tab[256 + c] = tab[512 + c];
    }
    uint32_t* tr = reinterpret_cast<uint32_t*>(dev_tab.data() + 512);
    for (uint64_t i = 0; i < ns * nc; i++) tr[i] = (uint32_t)trans[i] | ((uint32_t)(accept[trans[i]] + 1) << 16);
    CU_TRY(ctx, cudaSetDevice(ctx->device));
    anon_regex* rx = new (std::nothrow) anon_regex();
    if (!rx) return ANON_ERR_OOM;
    rx->ctx = ctx; rx->tab_bytes = (uint32_t)padded; rx->smem_bytes = (uint32_t)smem_need;
    rx->n_states = (int)ns; rx->n_classes = (int)nc; rx->n_patterns = (int)np; rx->max_match = (int)mm;
    if (cudaMalloc(&rx->d_tab, padded) != cudaSuccess) { cudaGetLastError(); delete rx; return ANON_ERR_OOM; }
    cudaError_t e = cudaMemcpyAsync(rx->d_tab, dev_tab.data(), padded, cudaMemcpyHostToDevice, ctx->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->stream);
    if (e == cudaSuccess)
    {   // the device's maximum, not this automaton's need: handles with different table sizes share the kernel
        cudaFuncAttributes fa;
        e = cudaFuncGetAttributes(&fa, regex_candidates_kernel);
        const long long max_dyn = (long long)ctx->smem_optin - (long long)fa.sharedSizeBytes;
        if (e == cudaSuccess && (long long)smem_need > max_dyn) { cudaFree(rx->d_tab); delete rx; return ANON_ERR_UNSUPPORTED; }
        if (e == cudaSuccess) e = cudaFuncSetAttribute(regex_candidates_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)max_dyn);
    }
    if (e == cudaSuccess)
        e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&rx->ctas_per_sm, regex_candidates_kernel, kThreads, smem_need);
    if (e != cudaSuccess) { cudaFree(rx->d_tab); delete rx; return cuda_fail(ctx, e, "anon_regex_load"); }
    if (rx->ctas_per_sm < 1) rx->ctas_per_sm = 1;
    *out = rx;
    return ANON_OK;
}

extern "C" void anon_regex_free(anon_regex* rx) {
    if (!rx) return;
    cudaSetDevice(rx->ctx->device);
    cudaFree(rx->d_tab);
    delete rx;
}

int regex_scan_impl(anon_ctx* ctx, WsCursor& ws, const anon_regex* rx, const uint8_t* d_text, size_t text_bytes,
                    const int64_t* d_rec_off, int32_t R, anon_span* d_spans, int32_t cap, int32_t* d_num)
{
    if (!ctx || !rx || R < 0 || cap < 0 || !d_num || !d_rec_off || (text_bytes > 0 && !d_text) || (cap > 0 && !d_spans))
        return ANON_ERR_INVALID_ARG;
    cudaStream_t st = ctx->stream;
    if (R == 0 || text_bytes == 0) { CU_TRY(ctx, cudaMemsetAsync(d_num, 0, 4, st)); return ANON_OK; }
    const long long nbytes = (long long)text_bytes;
    const long long n_tiles = (nbytes + kTile - 1) / kTile;
    uint16_t* cand = (uint16_t*)ws.take(((size_t)nbytes + 16) * 2);
    int* tile_rec = (int*)ws.take(((size_t)n_tiles + 1) * 4);
    int* rec_count = (int*)ws.take((size_t)R * 4);
    long long* rec_base = (long long*)ws.take((size_t)R * 8);
    long long* agg = (long long*)ws.take(scan::agg_bytes<long long>(R));
    if (!cand || !tile_rec || !rec_count || !rec_base || !agg) return ANON_ERR_OOM;
    ProfScope ps(ctx, PROF_DECODE, (double)nbytes * 7 + (double)R * 28, 8);
    const long long resident = (long long)ctx->sm_count * rx->ctas_per_sm;
    const unsigned grid = (unsigned)(n_tiles < resident ? n_tiles : resident);
    regex_tile_records_kernel<<<(unsigned)((n_tiles + 1 + kThreads - 1) / kThreads), kThreads, 0, st>>>((const long long*)d_rec_off, R, nbytes,
                                                                                                      n_tiles, tile_rec);
    regex_candidates_kernel<<<grid, kThreads, rx->smem_bytes, st>>>(rx->d_tab, rx->tab_bytes, rx->n_classes, rx->max_match, d_text, nbytes,
                                                                    (const long long*)d_rec_off, R, tile_rec, n_tiles, cand);
    const unsigned rblocks = (unsigned)((R + kThreads / 32 - 1) / (kThreads / 32));
    regex_select_kernel<<<(unsigned)((R + kSelWarps - 1) / kSelWarps), kSelWarps * 32, 0, st>>>(cand, (const long long*)d_rec_off, R, rec_count);
    CountIn cin{rec_count};
    scan::reduce_and_scan<long long, scan::SumI64>(cin, R, nullptr, agg, st);
    scan::apply<long long, scan::SumI64>(cin, BaseOut{rec_base}, R, nullptr, agg, st);
    regex_write_kernel<<<rblocks, kThreads, 0, st>>>(cand, (const long long*)d_rec_off, R, rec_base, rx->d_tab + 256, d_spans, (long long)cap);
    regex_finish_kernel<<<1, 1, 0, st>>>(agg + scan::num_tiles(R), (long long)cap, d_num, ctx->d_status);
    CU_LAUNCH_CHECK(ctx, "regex_scan");
    return ANON_OK;
}

int merge_spans_impl(anon_ctx* ctx, WsCursor& ws, const anon_span* d_ner, const int32_t* d_num_ner, int32_t ner_max,
                     const anon_span* d_rgx, const int32_t* d_num_rgx, int32_t rgx_max, anon_span* d_out, int32_t cap, int32_t* d_num_out)
{
    if (!ctx || ner_max < 0 || rgx_max < 0 || cap < 0 || !d_num_out || (ner_max > 0 && !d_ner) || (rgx_max > 0 && !d_rgx) ||
        (cap > 0 && !d_out))
        return ANON_ERR_INVALID_ARG;
    cudaStream_t st = ctx->stream;
    if (ner_max + (long long)rgx_max == 0) { CU_TRY(ctx, cudaMemsetAsync(d_num_out, 0, 4, st)); return ANON_OK; }
    const int n1 = ner_max > 0 ? ner_max : 1;
    uint8_t* keep = (uint8_t*)ws.take((size_t)n1);
    int* before = (int*)ws.take((size_t)n1 * 4);
    long long* kpos = (long long*)ws.take((size_t)n1 * 8);
    long long* agg = (long long*)ws.take(scan::agg_bytes<long long>(n1));
    if (!keep || !before || !kpos || !agg) return ANON_ERR_OOM;
    ProfScope ps(ctx, PROF_DECODE, ((double)ner_max + rgx_max) * 32, 5);
    if (ner_max > 0) {
        merge_flag_kernel<<<(unsigned)((ner_max + kThreads - 1) / kThreads), kThreads, 0, st>>>(d_ner, d_num_ner, ner_max, d_rgx, d_num_rgx,
                                                                                              rgx_max, keep, before);
        KeepIn kin{keep};
        scan::reduce_and_scan<long long, scan::SumI64>(kin, ner_max, d_num_ner, agg, st);
        scan::apply<long long, scan::SumI64>(kin, KeepOut{kpos}, ner_max, d_num_ner, agg, st);
    }
    const long long n = (long long)ner_max + rgx_max;
    merge_write_kernel<<<(unsigned)((n + kThreads - 1) / kThreads), kThreads, 0, st>>>(
        d_ner, d_num_ner, ner_max, d_rgx, d_num_rgx, rgx_max, keep, before, kpos, agg + scan::num_tiles(ner_max), d_out, (long long)cap,
        d_num_out, ctx->d_status);
    CU_LAUNCH_CHECK(ctx, "merge_spans");
    return ANON_OK;
}

extern "C" int anon_regex_scan(anon_ctx* ctx, const anon_regex* rx, const uint8_t* d_text, size_t text_bytes,
                               const int64_t* d_record_offsets, int32_t R, anon_span* d_spans, int32_t span_capacity,
                               int32_t* d_num_spans)
{
    if (!ctx) return ANON_ERR_INVALID_ARG;
    CU_TRY(ctx, cudaSetDevice(ctx->device));
    WsCursor ws = ws_begin(ctx);
    return regex_scan_impl(ctx, ws, rx, d_text, text_bytes, d_record_offsets, R, d_spans, span_capacity, d_num_spans);
}

extern "C" int anon_merge_spans(anon_ctx* ctx, const anon_span* d_ner_spans, const int32_t* d_num_ner, int32_t ner_max,
                                const anon_span* d_regex_spans, const int32_t* d_num_regex, int32_t regex_max,
                                anon_span* d_out_spans, int32_t capacity, int32_t* d_num_out)
{
    if (!ctx) return ANON_ERR_INVALID_ARG;
    CU_TRY(ctx, cudaSetDevice(ctx->device));
    WsCursor ws = ws_begin(ctx);
    return merge_spans_impl(ctx, ws, d_ner_spans, d_num_ner, ner_max, d_regex_spans, d_num_regex, regex_max, d_out_spans, capacity,
                            d_num_out);
}
