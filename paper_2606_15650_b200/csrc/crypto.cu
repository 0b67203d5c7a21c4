// crypto.cu -- A11 hash-cache dedup (K9), A12 HMAC-SHA256 (K10), A13 pseudonym write-back (K11).
// P:L43 (cache), P:L44 (HMAC-SHA256 slug, "[TYPE_slug]"), P:L50/L38 (referential integrity),
// P:L52 (entity, slug, full_hash rows); S8c O4; FIPS 180-4; RFC 2104.
//
// Determinism.  The sequential definition ("for i in order: hit or insert") is reproduced by a
// parallel protocol on one 64-bit word per slot:  [tag:32 | pending:1 | index:31].
//   probe    every span finds the slot of its string (full byte compare, never tag-only); the
//            first claimer CASes (tag, pending, i) into an empty slot and every later span of the
//            same string lowers the index with atomicMin, so the slot ends up naming the LOWEST
//            span index of each string that was not cached before the call.
//   classify span i is a miss iff its slot is pending and names i.  A transform-scan over
//            (miss, miss bytes, token bytes) gives dense uids in first-occurrence order, arena
//            offsets and out_offsets; the totals go to the host, which checks capacity BEFORE
//            anything persistent is written (otherwise the pending slots are rolled back to 0).
//   insert   one thread per NEW entity: copy bytes into the arena, HMAC, slot := (tag, 0, uid).
//   emit     every span reads its slot -> uid -> digest and writes its token.
#include "common.cuh"
#include "scan.cuh"

#include <algorithm>
#include <vector>
#include "sha256.cuh"

#include <new>

typedef unsigned long long u64;

struct anon_cache {
    anon_ctx* ctx = nullptr;
    uint64_t max_unique = 0, arena_bytes = 0, n_slots = 0;
    u64* d_table = nullptr;
    uint8_t* d_arena = nullptr;
    long long* d_entry_off = nullptr;   // [max_unique + 1]
    uint8_t* d_digests = nullptr;       // [max_unique, 32]
    uint64_t n_unique = 0, arena_used = 0, n_lookups = 0, n_hits = 0;
    // NEXT-5 (D21): call-granular recency.  epoch = number of anon_pseudonymize calls so far; d_last_use[uid] = epoch of the
    // last call that looked the entry up (allocated by anon_cache_track_use, NULL = not tracked)
    uint32_t* d_last_use = nullptr;
    uint32_t epoch = 0;
    bool key_bound = false;
    uint32_t ipad[8], opad[8];
};

struct PadStates { uint32_t ipad[8], opad[8]; };
struct TypeTable { uint8_t len[64]; alignas(4) char name[64][32]; int num; };

// ------------------------------------------------------------------------------------------------
// byte-stream helpers: read a message at any alignment as little-endian 32-bit words
// ------------------------------------------------------------------------------------------------
// bytes p[4j .. 4j+3], zero-filled past len.  Requires 4j < len.  Touches only aligned words that
// contain at least one byte of the message.
__device__ __forceinline__ uint32_t load_le_word(const uint8_t* p, int len, int j) {
    const uintptr_t addr = (uintptr_t)(p + 4 * j);
    const uint32_t a = (uint32_t)(addr & 3);
    const uint32_t* q = (const uint32_t*)(addr - a);
    const int remaining = len - 4 * j;
    uint32_t w = __ldg(q);
    if (a) {
        uint32_t hi = (remaining > (int)(4 - a)) ? __ldg(q + 1) : 0u;
        w = __funnelshift_r(w, hi, 8 * a);
    }
    if (remaining < 4) w &= (1u << (8 * remaining)) - 1u;
    return w;
}

// A byte string at any alignment read as consecutive little-endian 32-bit words, four at a time, through ALIGNED
// 16-byte loads (one LDG.128 per 16 bytes instead of up to eight 4-byte loads; a thread-per-span kernel pays one L1
// sector per load instruction, whatever its width).  Touches only aligned 16-byte chunks that contain at least one
// byte of the message.  Words past the end of the message are not defined: callers mask with tail_mask().
struct Words16 {
    const uint4* q; const uint8_t* end; uint4 prev; uint32_t wo, sh;
    __device__ __forceinline__ void init(const uint8_t* p, int len) {
        const uintptr_t addr = (uintptr_t)p;
        q = reinterpret_cast<const uint4*>(addr & ~(uintptr_t)15);
        end = p + len;
        wo = (uint32_t)(addr & 15) >> 2;
        sh = 8u * (uint32_t)(addr & 3);
        prev = len > 0 ? __ldg(q) : make_uint4(0u, 0u, 0u, 0u);
    }
    __device__ __forceinline__ void next4(uint32_t (&o)[4]) {
        q++;
        const uint4 cur = (reinterpret_cast<const uint8_t*>(q) < end) ? __ldg(q) : make_uint4(0u, 0u, 0u, 0u);
        // window of 8 words (prev, cur); wanted: words wo .. wo+4, then a byte funnel shift by sh
        uint32_t w0 = prev.x, w1 = prev.y, w2 = prev.z, w3 = prev.w, w4 = cur.x, w5 = cur.y, w6 = cur.z, w7 = cur.w;
        if (wo & 2u) { w0 = w2; w1 = w3; w2 = w4; w3 = w5; w4 = w6; w5 = w7; }
        if (wo & 1u) { w0 = w1; w1 = w2; w2 = w3; w3 = w4; w4 = w5; }
        o[0] = __funnelshift_r(w0, w1, sh); o[1] = __funnelshift_r(w1, w2, sh);
        o[2] = __funnelshift_r(w2, w3, sh); o[3] = __funnelshift_r(w3, w4, sh);
        prev = cur;
    }
};
// mask of word j of a len-byte message: all ones inside, partial on the last word, zero beyond
__device__ __forceinline__ uint32_t tail_mask(int len, int j) {
    const int rem = len - 4 * j;
    return rem >= 4 ? 0xFFFFFFFFu : (rem <= 0 ? 0u : (1u << (8 * rem)) - 1u);
}

// 64-bit hash of a byte string from four independent 32-bit lanes (one per word of a 16-byte chunk), each step
// acc = rotl(acc + w * P2, 13) * P1 -- two IMAD and one SHF per word instead of a 64-bit multiply chain per word (the probe
// kernel was instruction-bound with 34 % of its issue slots in IMAD; profiles/r02_pseudonym.md).  Words past the end of the
// message enter as zeros (only the last chunk is masked) and the length is mixed in at the end, so strings that differ only
// in trailing zero bytes still hash differently.  Only performance depends on the quality: equality is always decided by the
// full byte compare.
__device__ __forceinline__ u64 hash_bytes(const uint8_t* p, int len) {
    constexpr uint32_t P1 = 0x9E3779B1u, P2 = 0x85EBCA77u, P3 = 0xC2B2AE3Du, P4 = 0x27D4EB2Fu;
    uint32_t a0 = 0x243F6A88u, a1 = 0x85A308D3u, a2 = 0x13198A2Eu, a3 = 0x03707344u;
    const int nw = (len + 3) >> 2;
    Words16 ws; ws.init(p, len);
    for (int j = 0; j < nw; j += 4) {
        uint32_t w[4];
        ws.next4(w);
        if (j + 4 >= nw) {                            // last chunk: drop the bytes past the end
#pragma unroll
            for (int k = 0; k < 4; k++) w[k] &= tail_mask(len, j + k);
        }
        a0 = __funnelshift_l(a0 + w[0] * P2, a0 + w[0] * P2, 13) * P1;
        a1 = __funnelshift_l(a1 + w[1] * P2, a1 + w[1] * P2, 13) * P1;
        a2 = __funnelshift_l(a2 + w[2] * P2, a2 + w[2] * P2, 13) * P1;
        a3 = __funnelshift_l(a3 + w[3] * P2, a3 + w[3] * P2, 13) * P1;
    }
    uint32_t lo = __funnelshift_l(a0, a0, 1) + __funnelshift_l(a1, a1, 7) + __funnelshift_l(a2, a2, 12) + __funnelshift_l(a3, a3, 18) + (uint32_t)len;
    uint32_t hi = (a0 ^ __funnelshift_l(a1, a1, 15)) * P3 + (a2 ^ __funnelshift_l(a3, a3, 9)) * P4 + (uint32_t)len * P1;
    lo ^= lo >> 15; lo *= P2; lo ^= lo >> 13; lo *= P3; lo ^= lo >> 16;
    hi ^= hi >> 16; hi *= P1; hi ^= hi >> 13; hi *= P4; hi ^= hi >> 15;
    return ((u64)hi << 32) | lo;
}

__device__ __forceinline__ bool bytes_equal(const uint8_t* a, const uint8_t* b, int len) {
    const int nw = (len + 3) >> 2;
    Words16 wa, wb; wa.init(a, len); wb.init(b, len);
    for (int j = 0; j < nw; j += 4) {
        uint32_t x[4], y[4];
        wa.next4(x); wb.next4(y);
        uint32_t diff;
        if (j + 4 >= nw) {                            // last chunk: ignore the bytes past the end
            diff = 0;
#pragma unroll
            for (int k = 0; k < 4; k++) diff |= (x[k] ^ y[k]) & tail_mask(len, j + k);
        } else {
            diff = (x[0] ^ y[0]) | (x[1] ^ y[1]) | (x[2] ^ y[2]) | (x[3] ^ y[3]);
        }
        if (diff) return false;
    }
    return true;
}

// dst[0 .. len) = src[0 .. len) for byte strings at any alignment: up to three head bytes one by one until dst is word-aligned,
// then the source through aligned 16-byte loads (Words16) and 4-byte stores, the last 1-3 bytes one by one.  (The byte loop this
// replaces -- one LDG.U8 + one STG.U8 per byte -- was more than half of the insert kernel's time.)
__device__ __forceinline__ void copy_bytes(uint8_t* dst, const uint8_t* src, int len) {
    int head = (int)((4u - (uint32_t)(reinterpret_cast<uintptr_t>(dst) & 3)) & 3u);
    if (head > len) head = len;
    for (int k = 0; k < head; k++) dst[k] = src[k];
    dst += head; src += head; len -= head;
    if (len <= 0) return;
    uint32_t* d4 = reinterpret_cast<uint32_t*>(dst);
    const int nfull = len >> 2;
    Words16 ws; ws.init(src, len);
    for (int j = 0; j < nfull; j += 4) {
        uint32_t w[4];
        ws.next4(w);
#pragma unroll
        for (int k = 0; k < 4; k++) if (j + k < nfull) d4[j + k] = w[k];
    }
    for (int k = nfull << 2; k < len; k++) dst[k] = src[k];
}

__device__ __forceinline__ uint32_t slot_tag(u64 h) { uint32_t t = (uint32_t)(h >> 32); return t ? t : 1u; }
__device__ __forceinline__ u64 make_slot(uint32_t tag, uint32_t pending, uint32_t idx) {
    return ((u64)tag << 32) | ((u64)pending << 31) | idx;
}
__device__ __forceinline__ bool slot_pending(u64 v) { return (v >> 31) & 1ull; }
__device__ __forceinline__ uint32_t slot_index(u64 v) { return (uint32_t)(v & 0x7FFFFFFFull); }

// ------------------------------------------------------------------------------------------------
// K9 probe / insert-claim
// ------------------------------------------------------------------------------------------------
// The items of a block handed to its threads SORTED BY A WORK CLASS (0 .. 7; a counting sort in shared memory): returns the
// block-local index of the item this thread should take.  Thread-per-span kernels whose loops run once per 16-byte chunk or
// per SHA-256 block are as slow as the longest span of each warp; with span lengths spread over 7-128 bytes a warp of
// consecutive spans had 13 of 32 lanes active on average (profiles/r02_pseudonym.md).  Which thread takes which item must
// not matter for the result.  All threads of the block must call it.
#ifndef ANON_PROBE_SORT
#define ANON_PROBE_SORT 1
#endif
template <int BLOCK>
__device__ __forceinline__ int block_take_sorted(int cls) {
#if ANON_PROBE_SORT
    __shared__ int s_cnt[8];
    __shared__ uint16_t s_perm[BLOCK];
    if (threadIdx.x < 8) s_cnt[threadIdx.x] = 0;
    __syncthreads();
    const int rank = atomicAdd(&s_cnt[cls], 1);
    __syncthreads();
    int start = 0;
#pragma unroll
    for (int b = 0; b < 7; b++) start += b < cls ? s_cnt[b] : 0;
    s_perm[start + rank] = (uint16_t)threadIdx.x;
    __syncthreads();
    return (int)s_perm[threadIdx.x];
#else
    (void)cls;
    return (int)threadIdx.x;
#endif
}

// Six resident CTAs per SM (<= 40 registers, a few spilled words): with its spans in length-class order the kernel waits on its
// dependent random reads (slot -> first occurrence's offsets -> its bytes; ncu: 8 warps stalled on a long scoreboard per issue,
// 42 % of the warp slots occupied at 56 registers), and more warps in flight are worth more than the spills cost
// (50 M spans: 6.11 -> 5.95 ms per call; four CTAs 6.11, five 6.22, eight 6.00).
__global__ void __launch_bounds__(256, 6) cache_probe_kernel(
    const uint8_t* __restrict__ bytes, const long long* __restrict__ off, long long S,
    u64* table, u64 mask, const uint8_t* __restrict__ arena, const long long* __restrict__ entry_off,
    int* __restrict__ slot_of, int* d_full)
{
    // work class = 16-byte chunks of the span (the hash and the byte compare loop once per chunk); threads past the end go last
    long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    {
        const int my_len = i < S ? (int)(off[i + 1] - off[i]) : 0;
        const int cls = i < S ? min(max((my_len + 15) >> 4, 1), 8) - 1 : 7;
        i = (long long)blockIdx.x * blockDim.x + block_take_sorted<256>(cls);
    }
    if (i >= S) return;
    const long long o = off[i];
    const int len = (int)(off[i + 1] - o);
    const uint8_t* p = bytes + o;
    const u64 h = hash_bytes(p, len);
    const uint32_t tag = slot_tag(h);
    const u64 mine = make_slot(tag, 1u, (uint32_t)i);
    u64 slot = h & mask;
    for (u64 probes = 0; probes <= mask; probes++) {
        u64 v = *((volatile u64*)&table[slot]);
        if (v == 0) {
            v = atomicCAS(&table[slot], 0ull, mine);
            if (v == 0) { slot_of[i] = (int)slot; return; }
        }
        if ((uint32_t)(v >> 32) == tag) {
            bool eq;
            if (slot_pending(v)) {
                const long long r = slot_index(v);
                const long long ro = off[r];
                eq = (off[r + 1] - ro == len) && bytes_equal(p, bytes + ro, len);
            } else {
                const long long e = slot_index(v);
                const long long eo = entry_off[e];
                eq = (entry_off[e + 1] - eo == len) && bytes_equal(p, arena + eo, len);
            }
            if (eq) {
                if (slot_pending(v) && slot_index(v) > (uint32_t)i) atomicMin(&table[slot], mine);
                slot_of[i] = (int)slot;
                return;
            }
        }
        slot = (slot + 1) & mask;
    }
    slot_of[i] = -1;
    *d_full = 1;               // the probe's own flag (not the sticky status word: an earlier stage's CAPACITY is not "table full")
}

// ------------------------------------------------------------------------------------------------
// classify + scan functors
// ------------------------------------------------------------------------------------------------
// The scan evaluates its input twice (reduce pass, apply pass).  The first evaluation reads the span's slot -- a random 8-byte
// access per span -- and leaves the verdict in is_new[i]; the second (ClassifyAgain) reads that byte instead of the table.
struct ClassifyIn {
    const long long* off; const uint8_t* type; const int* slot_of; const u64* table;
    TypeTable tt; int slug_len; uint8_t* is_new_out;
    __device__ __forceinline__ scan::I64x3 operator()(long long i) const {
        const int s = slot_of[i];
        bool is_new = false;
        if (s >= 0) { u64 v = table[s]; is_new = slot_pending(v) && slot_index(v) == (uint32_t)i; }
        is_new_out[i] = is_new ? 1 : 0;
        int t = type ? type[i] : 0;
        if (t >= tt.num) t = tt.num - 1;
        return scan::I64x3{is_new ? 1 : 0, is_new ? off[i + 1] - off[i] : 0, 3 + tt.len[t] + slug_len};
    }
};
struct ClassifyAgain {
    const long long* off; const uint8_t* type; const uint8_t* is_new_in;
    TypeTable tt; int slug_len;
    __device__ __forceinline__ scan::I64x3 operator()(long long i) const {
        const bool is_new = is_new_in[i] != 0;
        int t = type ? type[i] : 0;
        if (t >= tt.num) t = tt.num - 1;
        return scan::I64x3{is_new ? 1 : 0, is_new ? off[i + 1] - off[i] : 0, 3 + tt.len[t] + slug_len};
    }
};
struct ClassifyOut {
    long long* out_off; uint8_t* hit; int* new_list; long long* entry_off;
    long long base_unique, arena_used, S;
    __device__ __forceinline__ void operator()(long long i, const scan::I64x3& ex, const scan::I64x3& v) const {
        out_off[i] = ex.c;
        if (hit) hit[i] = v.a ? 0 : 1;
        if (v.a) { new_list[ex.a] = (int)i; entry_off[base_unique + ex.a] = arena_used + ex.b; }
        if (i == S - 1) {
            out_off[S] = ex.c + v.c;
            entry_off[base_unique + ex.a + v.a] = arena_used + ex.b + v.b;
        }
    }
};

__global__ void __launch_bounds__(256) cache_rollback_kernel(long long S, const int* __restrict__ slot_of, u64* table) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= S) return;
    const int s = slot_of[i];
    if (s >= 0 && slot_pending(table[s])) table[s] = 0ull;
}

// ------------------------------------------------------------------------------------------------
// K10 HMAC-SHA256: one thread per message, W[16] ring in registers, pads precomputed on the host
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t bswap32(uint32_t x) { return __byte_perm(x, 0, 0x0123); }

__device__ __forceinline__ void hmac_message(const uint8_t* p, int len, const PadStates& ps, uint32_t out[8]) {
    uint32_t st[8];
#pragma unroll
    for (int k = 0; k < 8; k++) st[k] = ps.ipad[k];
    const int nblk = (len + 9 + 63) >> 6;
    uint32_t w[16];
    for (int b = 0; b < nblk; b++) {
#pragma unroll
        for (int t = 0; t < 16; t++) {
            const int j = b * 16 + t, pos = 4 * j;
            uint32_t x = 0;
            if (pos < len) x = load_le_word(p, len, j);
            if (pos <= len && len < pos + 4) x |= 0x80u << (8 * (len - pos));    // FIPS 180-4 §5.1.1
            w[t] = bswap32(x);
        }
        if (b == nblk - 1) w[15] = (uint32_t)(64 + len) * 8u;                     // bit length incl. the ipad block
        sha::compress(st, w);
    }
#pragma unroll
    for (int k = 0; k < 8; k++) w[k] = st[k];
    w[8] = 0x80000000u;
#pragma unroll
    for (int k = 9; k < 15; k++) w[k] = 0;
    w[15] = (64 + 32) * 8;
#pragma unroll
    for (int k = 0; k < 8; k++) out[k] = ps.opad[k];
    sha::compress(out, w);
}

// insert: thread r handles the r-th new entity of this call
__global__ void __launch_bounds__(128) cache_insert_kernel(
    const uint8_t* __restrict__ bytes, const long long* __restrict__ off, const int* __restrict__ new_list,
    long long n_new, long long base_unique, const int* __restrict__ slot_of, u64* table,
    uint8_t* arena, const long long* __restrict__ entry_off, uint32_t* digests, PadStates ps)
{
    // (sorting this kernel's items by SHA-256 block count like the probe's was measured: slower -- consecutive entities write
    // consecutive arena bytes, and the permutation breaks that: 6.80 against 6.64 ms for the whole call at 50 M spans)
    const long long r = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= n_new) return;
    const int i = new_list[r];
    const long long e = base_unique + r;
    const long long o = off[i];
    const int len = (int)(off[i + 1] - o);
    const uint8_t* p = bytes + o;
    uint8_t* dst = arena + entry_off[e];
    copy_bytes(dst, p, len);
    uint32_t d[8];
    hmac_message(p, len, ps, d);
    uint4* dg = (uint4*)(digests + e * 8);
    dg[0] = make_uint4(bswap32(d[0]), bswap32(d[1]), bswap32(d[2]), bswap32(d[3]));
    dg[1] = make_uint4(bswap32(d[4]), bswap32(d[5]), bswap32(d[6]), bswap32(d[7]));
    const int s = slot_of[i];
    table[s] = make_slot((uint32_t)(table[s] >> 32), 0u, (uint32_t)e);
}

// HMAC of every span, no dedup (anon_hmac_spans)
__global__ void __launch_bounds__(128) hmac_spans_kernel(
    const uint8_t* __restrict__ bytes, const long long* __restrict__ off, long long S, uint32_t* digests, PadStates ps)
{
    // work class = SHA-256 blocks of the inner hash (a warp is as slow as its longest message)
    long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    {
        const int cls = i < S ? min(((int)(off[i + 1] - off[i]) + 9 + 63) >> 6, 8) - 1 : 7;
        i = (long long)blockIdx.x * blockDim.x + block_take_sorted<128>(cls);
    }
    if (i >= S) return;
    const long long o = off[i];
    uint32_t d[8];
    hmac_message(bytes + o, (int)(off[i + 1] - o), ps, d);
    uint4* dg = (uint4*)(digests + i * 8);
    dg[0] = make_uint4(bswap32(d[0]), bswap32(d[1]), bswap32(d[2]), bswap32(d[3]));
    dg[1] = make_uint4(bswap32(d[4]), bswap32(d[5]), bswap32(d[6]), bswap32(d[7]));
}

// ------------------------------------------------------------------------------------------------
// K11 write-back
// ------------------------------------------------------------------------------------------------
// Each warp assembles the tokens of 32 consecutive spans -- a contiguous byte range of the output, since out_off is a
// prefix sum -- in shared memory (word-aligned with the global destination) and then copies the range with coalesced
// 4-byte stores; only the ragged first / last word of the range goes out byte by byte.  The type-name table is staged
// in shared memory once per CTA (lanes index it with different types).
constexpr int kEmitWarps = 8;
constexpr int kEmitMaxToken = 3 + 32 + 64;                 // '[' name '_' slug ']'
constexpr int kEmitWarpBytes = 32 * kEmitMaxToken + 8;     // + alignment slack

__global__ void __launch_bounds__(kEmitWarps * 32) emit_tokens_kernel(
    long long S, const int* __restrict__ slot_of, const u64* __restrict__ table, const uint8_t* __restrict__ type,
    const uint32_t* __restrict__ digests, const long long* __restrict__ out_off, uint8_t* out,
    long long* uid_out, uint8_t* dig_out, TypeTable tt, int slug_len, int* d_status, uint32_t* last_use, uint32_t epoch)
{
    __shared__ __align__(16) uint8_t s_tok[kEmitWarps][(kEmitWarpBytes + 15) / 16 * 16];
    __shared__ __align__(16) uint8_t s_name[64][32];
    __shared__ uint8_t s_len[64];
    // the table arrives as a kernel parameter (constant bank): a lane-varying index into it is serialised per distinct address
    // (ncu: ADU pipe 93 % busy when all 64 x 32 bytes were copied byte by byte), so only the num live names are copied, as words
    {
        const uint32_t* src = reinterpret_cast<const uint32_t*>(&tt.name[0][0]);
        uint32_t* dst = reinterpret_cast<uint32_t*>(&s_name[0][0]);
        for (int k = threadIdx.x; k < tt.num * 8; k += blockDim.x) dst[k] = src[k];
        if (threadIdx.x < tt.num) s_len[threadIdx.x] = tt.len[threadIdx.x];
    }
    __syncthreads();
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const long long i0 = ((long long)blockIdx.x * kEmitWarps + warp) * 32;
    if (i0 >= S) return;
    const long long i = i0 + lane;
    const bool live = i < S;
    const long long last = (i0 + 32 < S ? i0 + 32 : S);
    // `out` may sit at any byte address (a caller's sub-buffer): work in offsets relative to the 4-byte aligned address
    // just below it, so that "word-aligned" below means aligned in memory, not merely in the offset
    const long long mis = (long long)(reinterpret_cast<uintptr_t>(out) & 3);
    out -= mis;
    const long long b0 = out_off[i0] + mis, b1 = out_off[last] + mis;   // this warp's byte range of the output
    const long long base = b0 & ~3ll;                       // shared-memory offset 0 <-> global byte `base`
    uint8_t* buf = s_tok[warp];
    if (live) {
        const int s = slot_of[i];
        if (s >= 0) {
            const long long e = slot_index(table[s]);
            if (uid_out) uid_out[i] = e;
            if (last_use) last_use[e] = epoch;              // every writer of one call stores the same value
            const uint4* dg = (const uint4*)(digests + e * 8);
            const uint4 d0 = __ldg(dg), d1 = __ldg(dg + 1);
            if (dig_out) { uint4* q = (uint4*)(dig_out + i * 32); q[0] = d0; q[1] = d1; }
            int t = type ? type[i] : 0;
            if (t >= tt.num) { t = tt.num - 1; latch_status(d_status, ANON_ERR_UNSUPPORTED); }
            uint8_t* o = buf + (out_off[i] + mis - base);
            *o++ = '[';
            const int nl = s_len[t];
            for (int k = 0; k < nl; k++) *o++ = s_name[t][k];
            *o++ = '_';
            const uint32_t dw[8] = {d0.x, d0.y, d0.z, d0.w, d1.x, d1.y, d1.z, d1.w};   // little-endian words = digest bytes in order
#pragma unroll
            for (int k = 0; k < 8; k++) {                   // 8 hex characters per digest word, static register indexing
                if (8 * k >= slug_len) break;
#pragma unroll
                for (int j = 0; j < 8; j++) {
                    if (8 * k + j < slug_len) {
                        const uint32_t byte = (dw[k] >> (8 * (j >> 1))) & 0xFFu;
                        const uint32_t nib = (j & 1) ? (byte & 15u) : (byte >> 4);
                        o[8 * k + j] = (uint8_t)(nib < 10 ? '0' + nib : 'a' + (nib - 10));
                    }
                }
            }
            o[slug_len] = ']';
        }
    }
    __syncwarp();
    // coalesced copy of [b0, b1): whole words in between, bytes at the two ragged ends
    const long long w_lo = (b0 + 3) >> 2, w_hi = b1 >> 2;   // global word indices fully inside the range
    const uint32_t* bw = reinterpret_cast<const uint32_t*>(buf);
    uint32_t* ow = reinterpret_cast<uint32_t*>(out);
    if (w_lo <= w_hi) {
        for (long long w = w_lo + lane; w < w_hi; w += 32) ow[w] = bw[w - (base >> 2)];
        if (lane < 3) { const long long p = b0 + lane; if (p < (w_lo << 2) && p < b1) out[p] = buf[p - base]; }
        if (lane >= 29) { const long long p = (w_hi << 2) + (lane - 29); if (p < b1 && p >= (w_lo << 2)) out[p] = buf[p - base]; }
    } else {
        for (long long p = b0 + lane; p < b1; p += 32) out[p] = buf[p - base];
    }
}

// ------------------------------------------------------------------------------------------------
// host side
// ------------------------------------------------------------------------------------------------
static void host_sha256(const uint8_t* msg, size_t len, uint8_t out[32]) {
    uint32_t st[8];
    sha::init_state(st);
    const size_t padded = ((len + 9 + 63) / 64) * 64;
    for (size_t b = 0; b < padded; b += 64) {
        uint32_t w[16];
        for (int t = 0; t < 16; t++) {
            uint32_t x = 0;
            for (int k = 0; k < 4; k++) {
                size_t pos = b + 4 * t + k;
                uint8_t byte = pos < len ? msg[pos] : (pos == len ? 0x80 : 0);
                x = (x << 8) | byte;
            }
            w[t] = x;
        }
        if (b + 64 == padded) { w[14] = (uint32_t)(((uint64_t)len * 8) >> 32); w[15] = (uint32_t)((uint64_t)len * 8); }
        sha::compress(st, w);
    }
    for (int i = 0; i < 8; i++) { out[4 * i] = st[i] >> 24; out[4 * i + 1] = st[i] >> 16; out[4 * i + 2] = st[i] >> 8; out[4 * i + 3] = st[i]; }
}

// RFC 2104: K' = K (or SHA256(K) when longer than the block), zero-padded to 64 bytes; midstates of
// the (K' xor ipad) and (K' xor opad) blocks.
static void make_pads(const uint8_t* key, size_t key_len, PadStates* ps) {
    uint8_t k[64];
    memset(k, 0, sizeof k);
    if (key_len > 64) host_sha256(key, key_len, k);
    else if (key_len) memcpy(k, key, key_len);
    for (int which = 0; which < 2; which++) {
        uint32_t w[16];
        const uint8_t x = which ? 0x5c : 0x36;
        for (int t = 0; t < 16; t++)
            w[t] = ((uint32_t)(k[4 * t] ^ x) << 24) | ((uint32_t)(k[4 * t + 1] ^ x) << 16) |
                   ((uint32_t)(k[4 * t + 2] ^ x) << 8) | (uint32_t)(k[4 * t + 3] ^ x);
        uint32_t* st = which ? ps->opad : ps->ipad;
        sha::init_state(st);
        sha::compress(st, w);
    }
}

static int fill_type_table(const char* const* names, int num, TypeTable* tt) {
    memset(tt, 0, sizeof *tt);
    if (num < 1 || num > 64 || !names) return ANON_ERR_INVALID_ARG;
    for (int t = 0; t < num; t++) {
        if (!names[t]) return ANON_ERR_INVALID_ARG;
        size_t n = strlen(names[t]);
        if (n > 32) return ANON_ERR_UNSUPPORTED;
        tt->len[t] = (uint8_t)n;
        memcpy(tt->name[t], names[t], n);
    }
    tt->num = num;
    return ANON_OK;
}

extern "C" int anon_cache_create(anon_ctx* ctx, uint64_t max_unique, uint64_t key_arena_bytes, anon_cache** out) {
    if (!ctx || !out || max_unique == 0) return ANON_ERR_INVALID_ARG;
    if (max_unique > (1ull << 30)) return ANON_ERR_UNSUPPORTED;
    CU_TRY(ctx, cudaSetDevice(ctx->device));
    anon_cache* c = new (std::nothrow) anon_cache();
    if (!c) return ANON_ERR_OOM;
    c->ctx = ctx; c->max_unique = max_unique; c->arena_bytes = key_arena_bytes;
    uint64_t slots = 1024;
    while (slots < 2 * max_unique) slots <<= 1;
    c->n_slots = slots;
    cudaError_t e;
    if ((e = cudaMalloc(&c->d_table, slots * 8)) != cudaSuccess ||
        (e = cudaMalloc(&c->d_arena, key_arena_bytes + 16)) != cudaSuccess ||
        (e = cudaMalloc(&c->d_entry_off, (max_unique + 1) * 8)) != cudaSuccess ||
        (e = cudaMalloc(&c->d_digests, max_unique * 32)) != cudaSuccess) {
        anon_cache_destroy(c);
        cuda_fail(ctx, e, "cudaMalloc(cache)");
        return ANON_ERR_OOM;
    }
    CU_TRY(ctx, cudaMemsetAsync(c->d_table, 0, slots * 8, ctx->stream));
    CU_TRY(ctx, cudaMemsetAsync(c->d_entry_off, 0, 8, ctx->stream));
    CU_TRY(ctx, cudaStreamSynchronize(ctx->stream));
    *out = c;
    return ANON_OK;
}

extern "C" void anon_cache_destroy(anon_cache* c) {
    if (!c) return;
    cudaFree(c->d_table); cudaFree(c->d_arena); cudaFree(c->d_entry_off); cudaFree(c->d_digests); cudaFree(c->d_last_use);
    delete c;
}

extern "C" int anon_cache_clear(anon_cache* c) {
    if (!c) return ANON_ERR_INVALID_ARG;
    anon_ctx* ctx = c->ctx;
    CU_TRY(ctx, cudaSetDevice(ctx->device));
    CU_TRY(ctx, cudaMemsetAsync(c->d_table, 0, c->n_slots * 8, ctx->stream));
    c->n_unique = c->arena_used = c->n_lookups = c->n_hits = 0;
    c->epoch = 0;
    c->key_bound = false;
    return ANON_OK;
}

// ------------------------------------------------------------------------------------------------
// NEXT-5: bounded cache -- call-granular LRU eviction ("LRU cache"; reading D21)
// ------------------------------------------------------------------------------------------------
namespace {

struct EvictIn {
    const uint8_t* keep; const long long* entry_off;
    __device__ __forceinline__ scan::I64x3 operator()(long long e) const {
        const long long k = keep[e];
        return scan::I64x3{k, k ? entry_off[e + 1] - entry_off[e] : 0, 0};
    }
};
// survivors move to (new uid, new arena offset) in temporary arrays; one thread per old entry
struct EvictOut {
    const uint8_t* keep; const long long* entry_off; const uint8_t* arena; const uint32_t* digests; const uint32_t* last_use;
    long long* new_off; uint8_t* new_arena; uint32_t* new_digests; uint32_t* new_last_use; long long n;
    __device__ __forceinline__ void operator()(long long e, const scan::I64x3& ex, const scan::I64x3& v) const {
        if (v.a) {
            new_off[ex.a] = ex.b;
            const uint8_t* src = arena + entry_off[e];
            for (long long k = 0; k < v.b; k++) new_arena[ex.b + k] = src[k];
#pragma unroll
            for (int k = 0; k < 8; k++) new_digests[ex.a * 8 + k] = digests[e * 8 + k];
            new_last_use[ex.a] = last_use[e];
        }
        if (e == n - 1) new_off[ex.a + v.a] = ex.b + v.b;
    }
};

// rebuilds the table from the compacted entries: all strings are distinct, so the first empty slot of the probe sequence is it
__global__ void __launch_bounds__(256) cache_reinsert_kernel(const uint8_t* __restrict__ arena, const long long* __restrict__ entry_off,
                                                             long long n, u64* table, u64 mask)
{
    const long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= n) return;
    const long long o = entry_off[e];
    const u64 h = hash_bytes(arena + o, (int)(entry_off[e + 1] - o));
    const u64 mine = make_slot(slot_tag(h), 0u, (uint32_t)e);
    u64 slot = h & mask;
    while (atomicCAS(&table[slot], 0ull, mine) != 0ull) slot = (slot + 1) & mask;
}

}  // namespace

extern "C" int anon_cache_track_use(anon_cache* c, int enable) {
    if (!c) return ANON_ERR_INVALID_ARG;
    anon_ctx* ctx = c->ctx;
    CU_TRY(ctx, cudaSetDevice(ctx->device));
    CU_TRY(ctx, cudaStreamSynchronize(ctx->stream));
    if (!enable) { cudaFree(c->d_last_use); c->d_last_use = nullptr; return ANON_OK; }
    if (c->d_last_use) return ANON_OK;
    if (cudaMalloc(&c->d_last_use, c->max_unique * 4) != cudaSuccess) { cudaGetLastError(); return ANON_ERR_OOM; }
    CU_TRY(ctx, cudaMemset(c->d_last_use, 0, c->max_unique * 4));     // entries that predate tracking: oldest
    return ANON_OK;
}

extern "C" int anon_cache_evict(anon_cache* c, uint64_t keep, uint64_t* n_evicted) {
    if (!c) return ANON_ERR_INVALID_ARG;
    anon_ctx* ctx = c->ctx;
    if (n_evicted) *n_evicted = 0;
    if (!c->d_last_use) return ANON_ERR_UNSUPPORTED;                   // anon_cache_track_use first
    CU_TRY(ctx, cudaSetDevice(ctx->device));
    cudaStream_t st = ctx->stream;
    CU_TRY(ctx, cudaStreamSynchronize(st));
    const uint64_t n = c->n_unique;
    if (keep >= n) return ANON_OK;
    // which entries stay: the `keep` largest stamps, the lowest uids inside the cut-off stamp (host: n stamps, once per eviction)
    std::vector<uint32_t> stamp(n);
    CU_TRY(ctx, cudaMemcpy(stamp.data(), c->d_last_use, n * 4, cudaMemcpyDeviceToHost));
    std::vector<uint8_t> flag(n, 0);
    if (keep > 0) {
        std::vector<uint32_t> sorted(stamp);
        std::nth_element(sorted.begin(), sorted.begin() + (n - keep), sorted.end());
        const uint32_t cut = sorted[n - keep];                         // the keep-th largest stamp
        uint64_t above = 0;
        for (uint64_t e = 0; e < n; e++) above += stamp[e] > cut;
        uint64_t quota = keep - above;
        for (uint64_t e = 0; e < n; e++) {
            if (stamp[e] > cut) flag[e] = 1;
            else if (stamp[e] == cut && quota) { flag[e] = 1; quota--; }
        }
    }
    WsCursor ws = ws_begin(ctx);
    uint8_t* d_keep = (uint8_t*)ws.take(n);
    long long* new_off = (long long*)ws.take((keep + 1) * 8);
    uint8_t* new_arena = (uint8_t*)ws.take(c->arena_used + 16);
    uint32_t* new_dig = (uint32_t*)ws.take(keep * 32 + 32);
    uint32_t* new_use = (uint32_t*)ws.take(keep * 4 + 4);
    scan::I64x3* agg = (scan::I64x3*)ws.take(scan::agg_bytes<scan::I64x3>((long long)n));
    if (!d_keep || !new_off || !new_arena || !new_dig || !new_use || !agg) return ANON_ERR_OOM;
    CU_TRY(ctx, cudaMemcpyAsync(d_keep, flag.data(), n, cudaMemcpyHostToDevice, st));
    CU_TRY(ctx, cudaMemsetAsync(new_off, 0, 8, st));
    ProfScope prof(ctx, PROF_PSEUDO, 0.0, 4);
    EvictIn in{d_keep, c->d_entry_off};
    scan::reduce_and_scan<scan::I64x3, scan::SumI64x3>(in, (long long)n, nullptr, agg, st);
    scan::apply<scan::I64x3, scan::SumI64x3>(in, EvictOut{d_keep, c->d_entry_off, c->d_arena, (const uint32_t*)c->d_digests, c->d_last_use,
                                                          new_off, new_arena, new_dig, new_use, (long long)n},
                                             (long long)n, nullptr, agg, st);
    CU_LAUNCH_CHECK(ctx, "evict compaction");
    long long kept_bytes = 0;
    CU_TRY(ctx, cudaMemcpyAsync(&kept_bytes, new_off + keep, 8, cudaMemcpyDeviceToHost, st));
    CU_TRY(ctx, cudaStreamSynchronize(st));                            // also: flag[] has been consumed
    CU_TRY(ctx, cudaMemcpyAsync(c->d_entry_off, new_off, (keep + 1) * 8, cudaMemcpyDeviceToDevice, st));
    if (kept_bytes) CU_TRY(ctx, cudaMemcpyAsync(c->d_arena, new_arena, (size_t)kept_bytes, cudaMemcpyDeviceToDevice, st));
    if (keep) {
        CU_TRY(ctx, cudaMemcpyAsync(c->d_digests, new_dig, keep * 32, cudaMemcpyDeviceToDevice, st));
        CU_TRY(ctx, cudaMemcpyAsync(c->d_last_use, new_use, keep * 4, cudaMemcpyDeviceToDevice, st));
    }
    CU_TRY(ctx, cudaMemsetAsync(c->d_table, 0, c->n_slots * 8, st));
    if (keep) {
        cache_reinsert_kernel<<<(unsigned)((keep + 255) / 256), 256, 0, st>>>(c->d_arena, c->d_entry_off, (long long)keep, c->d_table,
                                                                             c->n_slots - 1);
        CU_LAUNCH_CHECK(ctx, "cache_reinsert_kernel");
    }
    CU_TRY(ctx, cudaStreamSynchronize(st));
    c->n_unique = keep;
    c->arena_used = (uint64_t)kept_bytes;
    if (n_evicted) *n_evicted = n - keep;
    return ANON_OK;
}

extern "C" int anon_cache_stats(anon_cache* c, uint64_t* n_unique, uint64_t* n_lookups, uint64_t* n_hits) {
    if (!c) return ANON_ERR_INVALID_ARG;
    CU_TRY(c->ctx, cudaStreamSynchronize(c->ctx->stream));
    if (n_unique) *n_unique = c->n_unique;
    if (n_lookups) *n_lookups = c->n_lookups;
    if (n_hits) *n_hits = c->n_hits;
    return ANON_OK;
}

extern "C" int64_t anon_cache_entry(anon_cache* c, uint64_t uid, uint8_t* h_bytes, size_t cap, uint8_t* h_digest) {
    if (!c) return ANON_ERR_INVALID_ARG;
    anon_ctx* ctx = c->ctx;
    CU_TRY(ctx, cudaStreamSynchronize(ctx->stream));
    if (uid >= c->n_unique) return ANON_ERR_INVALID_ARG;
    long long o[2];
    CU_TRY(ctx, cudaMemcpy(o, c->d_entry_off + uid, 16, cudaMemcpyDeviceToHost));
    const int64_t len = o[1] - o[0];
    if (h_bytes && len > 0 && cap > 0)
        CU_TRY(ctx, cudaMemcpy(h_bytes, c->d_arena + o[0], (size_t)len < cap ? (size_t)len : cap, cudaMemcpyDeviceToHost));
    if (h_digest) CU_TRY(ctx, cudaMemcpy(h_digest, c->d_digests + uid * 32, 32, cudaMemcpyDeviceToHost));
    return len;
}

extern "C" int anon_cache_export(anon_cache* c, uint8_t* h_bytes, size_t bytes_capacity, int64_t* h_offsets, uint8_t* h_digests,
                                 uint64_t* n_unique, uint64_t* n_bytes)
{
    if (!c) return ANON_ERR_INVALID_ARG;
    anon_ctx* ctx = c->ctx;
    CU_TRY(ctx, cudaSetDevice(ctx->device));
    CU_TRY(ctx, cudaStreamSynchronize(ctx->stream));
    if (n_unique) *n_unique = c->n_unique;
    if (n_bytes) *n_bytes = c->arena_used;
    if (h_bytes && bytes_capacity < c->arena_used) return ANON_ERR_CAPACITY;
    if (h_offsets) CU_TRY(ctx, cudaMemcpy(h_offsets, c->d_entry_off, (c->n_unique + 1) * 8, cudaMemcpyDeviceToHost));
    if (h_bytes && c->arena_used) CU_TRY(ctx, cudaMemcpy(h_bytes, c->d_arena, c->arena_used, cudaMemcpyDeviceToHost));
    if (h_digests && c->n_unique) CU_TRY(ctx, cudaMemcpy(h_digests, c->d_digests, c->n_unique * 32, cudaMemcpyDeviceToHost));
    return ANON_OK;
}

int pseudonymize_impl(anon_ctx* ctx, WsCursor& ws, anon_cache* c, const uint8_t* d_bytes, const int64_t* d_off,
                      const uint8_t* d_type, int64_t S, const uint8_t* key, size_t key_len, int32_t slug_len,
                      const char* const* type_names, int32_t num_types, uint8_t* d_out, size_t out_cap,
                      int64_t* d_out_off, uint8_t* d_hit, int64_t* d_uid, uint8_t* d_digests,
                      int64_t* total_out_bytes)
{
    if (!ctx || !c || c->ctx != ctx || S < 0 || !d_off || !d_out_off || (!key && key_len) || slug_len < 0 || slug_len > 64)
        return ANON_ERR_INVALID_ARG;
    if (S > 0 && (!d_bytes || !d_out)) return ANON_ERR_INVALID_ARG;
    // uint4 stores of the per-span digests: 16-byte alignment is part of the ABI (include/anonshield.h)
    if (d_digests && (reinterpret_cast<uintptr_t>(d_digests) & 15)) return ANON_ERR_INVALID_ARG;
    if (S >= (1ll << 31)) return ANON_ERR_UNSUPPORTED;
    TypeTable tt;
    int rc = fill_type_table(type_names, num_types, &tt);
    if (rc) return rc;
    PadStates ps;
    make_pads(key, key_len, &ps);
    if (c->key_bound) {
        if (memcmp(ps.ipad, c->ipad, 32) || memcmp(ps.opad, c->opad, 32)) return ANON_ERR_KEY_MISMATCH;
    }
    cudaStream_t st = ctx->stream;
    if (total_out_bytes) *total_out_bytes = 0;
    if (S == 0) {
        CU_TRY(ctx, cudaMemsetAsync(d_out_off, 0, 8, st));
        if (!c->key_bound) { memcpy(c->ipad, ps.ipad, 32); memcpy(c->opad, ps.opad, 32); c->key_bound = true; }
        return ANON_OK;
    }
    int* slot_of = (int*)ws.take((size_t)S * 4);
    int* new_list = (int*)ws.take((size_t)S * 4);
    scan::I64x3* agg = (scan::I64x3*)ws.take(scan::agg_bytes<scan::I64x3>(S));
    uint8_t* is_new = (uint8_t*)ws.take((size_t)S);
    if (!slot_of || !new_list || !agg || !is_new) return ANON_ERR_OOM;
    const long long* off = (const long long*)d_off;
    const unsigned nb256 = (unsigned)((S + 255) / 256);
    ProfScope prof(ctx, PROF_PSEUDO, 0.0, 6);

    int* d_full = ctx->d_status + 16;
    CU_TRY(ctx, cudaMemsetAsync(d_full, 0, 4, st));
    cache_probe_kernel<<<nb256, 256, 0, st>>>(d_bytes, off, S, c->d_table, c->n_slots - 1, c->d_arena,
                                               c->d_entry_off, slot_of, d_full);
    CU_LAUNCH_CHECK(ctx, "cache_probe_kernel");
    ClassifyIn in{off, d_type, slot_of, c->d_table, tt, slug_len, is_new};
    scan::reduce_and_scan<scan::I64x3, scan::SumI64x3>(in, S, nullptr, agg, st);
    CU_LAUNCH_CHECK(ctx, "classify scan");
    scan::I64x3* h_tot = (scan::I64x3*)ctx->h_pinned;
    int* h_status = (int*)(ctx->h_pinned + 64);
    CU_TRY(ctx, cudaMemcpyAsync(h_tot, agg + scan::num_tiles(S), sizeof(scan::I64x3), cudaMemcpyDeviceToHost, st));
    CU_TRY(ctx, cudaMemcpyAsync(h_status, d_full, 4, cudaMemcpyDeviceToHost, st));
    CU_TRY(ctx, cudaStreamSynchronize(st));
    const long long n_new = h_tot->a, new_bytes = h_tot->b, out_bytes = h_tot->c;
    if (total_out_bytes) *total_out_bytes = out_bytes;
    const bool table_full = (*h_status != 0);
    if (table_full || c->n_unique + (uint64_t)n_new > c->max_unique ||
        c->arena_used + (uint64_t)new_bytes > c->arena_bytes || (uint64_t)out_bytes > out_cap) {
        cache_rollback_kernel<<<nb256, 256, 0, st>>>(S, slot_of, c->d_table);
        CU_TRY(ctx, cudaStreamSynchronize(st));
        return ANON_ERR_CAPACITY;
    }
    ClassifyOut outf{(long long*)d_out_off, d_hit, new_list, c->d_entry_off, (long long)c->n_unique,
                     (long long)c->arena_used, S};
    ClassifyAgain in2{off, d_type, is_new, tt, slug_len};
    scan::apply<scan::I64x3, scan::SumI64x3>(in2, outf, S, nullptr, agg, st);
    CU_LAUNCH_CHECK(ctx, "classify apply");
    if (n_new > 0) {
        cache_insert_kernel<<<(unsigned)((n_new + 127) / 128), 128, 0, st>>>(
            d_bytes, off, new_list, n_new, (long long)c->n_unique, slot_of, c->d_table, c->d_arena,
            c->d_entry_off, (uint32_t*)c->d_digests, ps);
        CU_LAUNCH_CHECK(ctx, "cache_insert_kernel");
    }
    emit_tokens_kernel<<<nb256, kEmitWarps * 32, 0, st>>>(S, slot_of, c->d_table, d_type, (const uint32_t*)c->d_digests,
                                               (const long long*)d_out_off, d_out, (long long*)d_uid, d_digests,
                                               tt, slug_len, ctx->d_status, c->d_last_use, c->epoch + 1);
    CU_LAUNCH_CHECK(ctx, "emit_tokens_kernel");
    c->epoch++;
    if (!c->key_bound) { memcpy(c->ipad, ps.ipad, 32); memcpy(c->opad, ps.opad, 32); c->key_bound = true; }
    c->n_unique += (uint64_t)n_new;
    c->arena_used += (uint64_t)new_bytes;
    c->n_lookups += (uint64_t)S;
    c->n_hits += (uint64_t)(S - n_new);
    return ANON_OK;
}

extern "C" int anon_pseudonymize(anon_ctx* ctx, anon_cache* cache, const uint8_t* d_span_bytes,
                                 const int64_t* d_span_offsets, const uint8_t* d_span_type, int64_t S,
                                 const uint8_t* key, size_t key_len, int32_t slug_len,
                                 const char* const* type_names, int32_t num_types, uint8_t* d_out_tokens,
                                 size_t out_capacity, int64_t* d_out_offsets, uint8_t* d_hit, int64_t* d_uid,
                                 uint8_t* d_digests)
{
    if (!ctx) return ANON_ERR_INVALID_ARG;
    CU_TRY(ctx, cudaSetDevice(ctx->device));
    WsCursor ws = ws_begin(ctx);
    return pseudonymize_impl(ctx, ws, cache, d_span_bytes, d_span_offsets, d_span_type, S, key, key_len, slug_len,
                             type_names, num_types, d_out_tokens, out_capacity, d_out_offsets, d_hit, d_uid,
                             d_digests, nullptr);
}

extern "C" int anon_hmac_spans(anon_ctx* ctx, const uint8_t* d_span_bytes, const int64_t* d_span_offsets, int64_t S,
                               const uint8_t* key, size_t key_len, uint8_t* d_digests)
{
    if (!ctx || S < 0 || !d_span_offsets || (S > 0 && (!d_digests || !d_span_bytes)) || (!key && key_len)) return ANON_ERR_INVALID_ARG;
    if (reinterpret_cast<uintptr_t>(d_digests) & 15) return ANON_ERR_INVALID_ARG;      // uint4 stores
    CU_TRY(ctx, cudaSetDevice(ctx->device));
    if (S == 0) return ANON_OK;
    PadStates ps;
    make_pads(key, key_len, &ps);
    ProfScope prof(ctx, PROF_PSEUDO, 0.0, 1);
    hmac_spans_kernel<<<(unsigned)((S + 127) / 128), 128, 0, ctx->stream>>>(
        d_span_bytes, (const long long*)d_span_offsets, S, (uint32_t*)d_digests, ps);
    CU_LAUNCH_CHECK(ctx, "hmac_spans_kernel");
    return ANON_OK;
}
