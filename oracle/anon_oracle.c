/*
 * anon_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, single-threaded CPU oracle for the integer half of the AnonShield hot
 * path (arxiv/paper_2606_15650): SHA-256, HMAC-SHA256, entity dedup through a cache,
 * pseudonym write-back.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may call this.  It shares no code with the CUDA
 * path under paper_2606_15650_b200/csrc/.
 *
 * Passages followed:
 *   PAPER.md L44 (§II stage 3): "Each entity is replaced by an HMAC-SHA256 slug computed
 *     with an operator-defined secret key. The slug length is configurable from 0 to 64
 *     hexadecimal characters ..., and the entity type is preserved as a prefix, e.g.
 *     100.111.20.23 -> [IP_ADDRESS_48624b5cdc]."
 *   PAPER.md L43 (§II stage 2): "an LRU cache to amortise repeated lookups across records".
 *   PAPER.md L50 (Fig. 1 caption) / L38: same entity + same key => same pseudonym.
 *   PAPER.md L52 (§II stage 4): mapping row keeps slug_name and full_hash.
 *   SURVEY.md §8(c) O4 (readings S12-S19: raw bytes hashed, type not hashed, first
 *     slug_len lower-case hex chars, "[TYPE_]" for slug_len 0, no eviction).
 *   FIPS 180-4 §4.1.2, §4.2.2, §5.1.1, §5.3.3, §6.2 (SHA-256); RFC 2104 §2 (HMAC).
 *
 * Pins (tests/test_oracle_crypto.py): FIPS 180-4 / RFC 4231 vectors in tests/golden/,
 * Python hashlib/hmac on every padding boundary, constants re-derived from the cube /
 * square roots of the primes, dict-based brute-force dedup.
 */
#include <stdint.h>
#include <stddef.h>
#include <stdlib.h>
#include <string.h>

/* ---- FIPS 180-4 §4.2.2 / §5.3.3: constants from the fractional parts of the cube roots
 * (K) of the first 64 primes and of the square roots (H0) of the first 8 primes.
 * Computed here with exact integer arithmetic instead of a pasted table. ---- */
static uint32_t K256[64];
static uint32_t H256[8];
static int consts_ready = 0;

typedef unsigned __int128 u128;

/* floor(frac(n^(1/r)) * 2^32) for r = 2 or 3: binary search the largest 64-bit x with
 * x^r <= n * 2^(32 r), then keep the low 32 bits (the integer part is above bit 32). */
static uint32_t frac_root_bits(uint32_t n, int r)
{
    uint64_t lo = 0, hi = (uint64_t)1 << 40; /* n < 2^9 so the root < 2^3 * 2^32 */
    while (hi - lo > 1) {
        uint64_t mid = lo + (hi - lo) / 2;
        u128 p = (u128)mid * mid;                 /* < 2^80 */
        int le;
        if (r == 2) le = p <= ((u128)n << 64);
        else        le = p * mid <= ((u128)n << 96); /* mid^3 < 2^120: no overflow */
        if (le) lo = mid; else hi = mid;
    }
    return (uint32_t)(lo & 0xffffffffu);
}

static void init_consts(void)
{
    if (consts_ready) return;
    uint32_t primes[64];
    int np = 0;
    for (uint32_t c = 2; np < 64; c++) {
        int is_p = 1;
        for (uint32_t d = 2; d * d <= c; d++) if (c % d == 0) { is_p = 0; break; }
        if (is_p) primes[np++] = c;
    }
    for (int i = 0; i < 64; i++) K256[i] = frac_root_bits(primes[i], 3);
    for (int i = 0; i < 8; i++)  H256[i] = frac_root_bits(primes[i], 2);
    consts_ready = 1;
}

void oracle_sha256_constants(uint32_t *k64, uint32_t *h8)
{
    init_consts();
    memcpy(k64, K256, sizeof K256);
    memcpy(h8, H256, sizeof H256);
}

/* ---- FIPS 180-4 §4.1.2 functions ---- */
static uint32_t rotr(uint32_t x, int n) { return (x >> n) | (x << (32 - n)); }
static uint32_t Ch(uint32_t x, uint32_t y, uint32_t z)  { return (x & y) ^ (~x & z); }
static uint32_t Maj(uint32_t x, uint32_t y, uint32_t z) { return (x & y) ^ (x & z) ^ (y & z); }
static uint32_t BSIG0(uint32_t x) { return rotr(x, 2) ^ rotr(x, 13) ^ rotr(x, 22); }
static uint32_t BSIG1(uint32_t x) { return rotr(x, 6) ^ rotr(x, 11) ^ rotr(x, 25); }
static uint32_t SSIG0(uint32_t x) { return rotr(x, 7) ^ rotr(x, 18) ^ (x >> 3); }
static uint32_t SSIG1(uint32_t x) { return rotr(x, 17) ^ rotr(x, 19) ^ (x >> 10); }

/* FIPS 180-4 §6.2.2: one 512-bit block. */
static void sha256_block(uint32_t H[8], const uint8_t M[64])
{
    uint32_t W[64];
    for (int t = 0; t < 16; t++)
        W[t] = ((uint32_t)M[4 * t] << 24) | ((uint32_t)M[4 * t + 1] << 16) |
               ((uint32_t)M[4 * t + 2] << 8) | (uint32_t)M[4 * t + 3];
    for (int t = 16; t < 64; t++)
        W[t] = SSIG1(W[t - 2]) + W[t - 7] + SSIG0(W[t - 15]) + W[t - 16];
    uint32_t a = H[0], b = H[1], c = H[2], d = H[3], e = H[4], f = H[5], g = H[6], h = H[7];
    for (int t = 0; t < 64; t++) {
        uint32_t T1 = h + BSIG1(e) + Ch(e, f, g) + K256[t] + W[t];
        uint32_t T2 = BSIG0(a) + Maj(a, b, c);
        h = g; g = f; f = e; e = d + T1; d = c; c = b; b = a; a = T1 + T2;
    }
    H[0] += a; H[1] += b; H[2] += c; H[3] += d; H[4] += e; H[5] += f; H[6] += g; H[7] += h;
}

/* FIPS 180-4 §5.1.1 padding + §6.2: the message is materialised padded, then hashed
 * block by block (no streaming state: slow and obvious). */
void oracle_sha256(const uint8_t *msg, uint64_t len, uint8_t out[32])
{
    init_consts();
    uint64_t padded = ((len + 9 + 63) / 64) * 64;
    uint8_t *buf = (uint8_t *)calloc(padded, 1);
    if (len) memcpy(buf, msg, len);
    buf[len] = 0x80;
    uint64_t bits = len * 8;
    for (int i = 0; i < 8; i++) buf[padded - 1 - i] = (uint8_t)(bits >> (8 * i));
    uint32_t H[8];
    memcpy(H, H256, sizeof H);
    for (uint64_t off = 0; off < padded; off += 64) sha256_block(H, buf + off);
    for (int i = 0; i < 8; i++) {
        out[4 * i] = (uint8_t)(H[i] >> 24); out[4 * i + 1] = (uint8_t)(H[i] >> 16);
        out[4 * i + 2] = (uint8_t)(H[i] >> 8); out[4 * i + 3] = (uint8_t)H[i];
    }
    free(buf);
}

/* RFC 2104 §2: H((K' xor opad) || H((K' xor ipad) || m)), B = 64, K' = H(K) if |K| > B. */
void oracle_hmac_sha256(const uint8_t *key, uint64_t key_len,
                        const uint8_t *msg, uint64_t len, uint8_t out[32])
{
    uint8_t kp[64];
    memset(kp, 0, 64);
    if (key_len > 64) oracle_sha256(key, key_len, kp);
    else if (key_len) memcpy(kp, key, key_len);
    uint8_t *inner = (uint8_t *)malloc(64 + len);
    for (int i = 0; i < 64; i++) inner[i] = kp[i] ^ 0x36;
    if (len) memcpy(inner + 64, msg, len);
    uint8_t ih[32];
    oracle_sha256(inner, 64 + len, ih);
    free(inner);
    uint8_t outer[96];
    for (int i = 0; i < 64; i++) outer[i] = kp[i] ^ 0x5c;
    memcpy(outer + 64, ih, 32);
    oracle_sha256(outer, 96, out);
}

/* Batch HMAC over CSR messages (no dedup): digests[i] = HMAC(key, bytes[off[i]:off[i+1]]). */
void oracle_hmac_batch(const uint8_t *key, uint64_t key_len, const uint8_t *bytes,
                       const int64_t *off, int64_t n, uint8_t *digests)
{
    for (int64_t i = 0; i < n; i++)
        oracle_hmac_sha256(key, key_len, bytes + off[i], (uint64_t)(off[i + 1] - off[i]),
                           digests + 32 * i);
}

/* ---- the cache M : byte-string -> (digest, uid).  A chained hash map
 * with full byte compare; the bucket hash only picks a chain and never decides equality. */
typedef struct entry {
    struct entry *next;
    uint8_t *bytes;
    uint64_t len;
    int64_t uid;
    uint8_t digest[32];
} entry;

typedef struct {
    entry **buckets;
    uint64_t nbuckets;
    int64_t n_unique, n_lookups, n_hits;
    uint8_t *key;
    uint64_t key_len;
    entry **by_uid;
    int64_t by_uid_cap;
} oracle_cache;

oracle_cache *oracle_cache_create(uint64_t nbuckets)
{
    oracle_cache *c = (oracle_cache *)calloc(1, sizeof *c);
    c->nbuckets = nbuckets ? nbuckets : 1;
    c->buckets = (entry **)calloc(c->nbuckets, sizeof(entry *));
    return c;
}

void oracle_cache_destroy(oracle_cache *c)
{
    if (!c) return;
    for (uint64_t b = 0; b < c->nbuckets; b++)
        for (entry *e = c->buckets[b]; e;) { entry *n = e->next; free(e->bytes); free(e); e = n; }
    free(c->buckets); free(c->key); free(c->by_uid); free(c);
}

void oracle_cache_stats(const oracle_cache *c, int64_t *n_unique, int64_t *n_lookups, int64_t *n_hits)
{
    *n_unique = c->n_unique; *n_lookups = c->n_lookups; *n_hits = c->n_hits;
}

/* Export of entry uid: length, then bytes and digest into caller buffers (PAPER.md L52 row:
 * original_name, full_hash).  Returns the length, or -1 for an unknown uid. */
int64_t oracle_cache_entry(const oracle_cache *c, int64_t uid, uint8_t *bytes_out, uint64_t cap, uint8_t digest_out[32])
{
    if (uid < 0 || uid >= c->n_unique) return -1;
    const entry *e = c->by_uid[uid];
    if (bytes_out && e->len <= cap && e->len) memcpy(bytes_out, e->bytes, e->len);
    if (digest_out) memcpy(digest_out, e->digest, 32);
    return (int64_t)e->len;
}

static uint64_t bucket_of(const oracle_cache *c, const uint8_t *p, uint64_t n)
{
    uint64_t h = 1469598103934665603ull;
    for (uint64_t i = 0; i < n; i++) h = (h ^ p[i]) * 1099511628211ull;
    return h % c->nbuckets;
}

/*
 * O4 loop.  Returns 0, -1 if the cache is bound to another key, -2 on a bad argument,
 * -3 if out_capacity is too small (out_offsets[] is still complete).
 * out_offsets[S+1] = exclusive prefix sum of 3 + |type_names[type]| + slug_len.
 */
int oracle_pseudonymize(oracle_cache *c, const uint8_t *span_bytes, const int64_t *span_off,
                        const uint8_t *span_type, int64_t S, const uint8_t *key, uint64_t key_len,
                        int32_t slug_len, const char *const *type_names, int32_t num_types,
                        uint8_t *out_tokens, uint64_t out_capacity, int64_t *out_offsets,
                        uint8_t *hit, int64_t *uid, uint8_t *digests)
{
    static const char hexd[] = "0123456789abcdef";
    if (slug_len < 0 || slug_len > 64 || S < 0 || num_types < 1) return -2;
    if (!c->key) {
        c->key = (uint8_t *)malloc(key_len ? key_len : 1);
        if (key_len) memcpy(c->key, key, key_len);
        c->key_len = key_len;
    } else if (c->key_len != key_len || (key_len && memcmp(c->key, key, key_len) != 0)) {
        return -1;
    }
    int64_t pos = 0;
    int overflow = 0;
    for (int64_t i = 0; i < S; i++) {
        const uint8_t *e = span_bytes + span_off[i];
        uint64_t len = (uint64_t)(span_off[i + 1] - span_off[i]);
        uint64_t b = bucket_of(c, e, len);
        entry *f = c->buckets[b];
        while (f && !(f->len == len && (len == 0 || memcmp(f->bytes, e, len) == 0))) f = f->next;
        c->n_lookups++;
        int h = 1;
        if (!f) {
            h = 0;
            f = (entry *)calloc(1, sizeof *f);
            f->bytes = (uint8_t *)malloc(len ? len : 1);
            if (len) memcpy(f->bytes, e, len);
            f->len = len;
            f->uid = c->n_unique;
            oracle_hmac_sha256(key, key_len, e, len, f->digest);
            f->next = c->buckets[b];
            c->buckets[b] = f;
            if (c->n_unique >= c->by_uid_cap) {
                c->by_uid_cap = c->by_uid_cap ? 2 * c->by_uid_cap : 1024;
                c->by_uid = (entry **)realloc(c->by_uid, (size_t)c->by_uid_cap * sizeof(entry *));
            }
            c->by_uid[c->n_unique++] = f;
        } else {
            c->n_hits++;
        }
        if (hit) hit[i] = (uint8_t)h;
        if (uid) uid[i] = f->uid;
        if (digests) memcpy(digests + 32 * i, f->digest, 32);
        int t = span_type ? span_type[i] : 0;
        if (t >= num_types) return -2;
        const char *name = type_names[t];
        uint64_t nl = strlen(name);
        uint64_t tok = 3 + nl + (uint64_t)slug_len;
        out_offsets[i] = pos;
        if ((uint64_t)pos + tok <= out_capacity && out_tokens) {
            uint8_t *o = out_tokens + pos;
            *o++ = '[';
            memcpy(o, name, nl); o += nl;
            *o++ = '_';
            for (int k = 0; k < slug_len; k++) {
                uint8_t byte = f->digest[k / 2];
                *o++ = (uint8_t)hexd[(k % 2 == 0) ? (byte >> 4) : (byte & 15)];
            }
            *o++ = ']';
        } else {
            overflow = 1;
        }
        pos += (int64_t)tok;
    }
    out_offsets[S] = pos;
    return overflow ? -3 : 0;
}
