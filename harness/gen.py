"""Seeded synthetic inputs for the five BASELINE.json configs.

This module holds NONE of the method's arithmetic: it only draws parameters, token ids,
record text and entity strings, and lays them out.  Both the oracle and the CUDA path are
fed from here (they share data, never code).  Everything is numpy on the host; seeds are
260615650 + config number.

Stand-in statement: the paper measures on D1/D1C/D3 (public in its repository, not in this
container) and D2 (private) -- PAPER.md L61-L91.  The records below take D2's record count
(70,951), total size (~550 MB) and mean record size, and D3's Zipf-like entity reuse, and
stand in for them; no item of those datasets is reproduced.
"""
import numpy as np

SEED_BASE = 260615650

# ---- model shapes (BASELINE.json configs[0..3]) -------------------------------------------
DESCS = {
    "tiny": dict(layers=2, hidden=128, heads=2, ffn=512, vocab=8192, num_labels=9, max_pos=512,
                 ln_eps=1e-5, dtype=0),
    "base": dict(layers=12, hidden=768, heads=12, ffn=3072, vocab=30522, num_labels=13, max_pos=512,
                 ln_eps=1e-5, dtype=1),
    "large": dict(layers=24, hidden=1024, heads=16, ffn=4096, vocab=250002, num_labels=13,
                  max_pos=512, ln_eps=1e-5, dtype=1),
}
# NEXT-3: ModernBERT-shaped variants (reading D20): arch 1 = pre-LN, RoPE, GeGLU (W_i is [2 ffn, hidden]), local window 128
# in every layer that is not a multiple of global_every, no biases.  "base_modern" has ModernBERT-base's published sizes.
_MODERN = dict(arch=1, local_window=128, global_every=3, rope_theta_global=160000.0, rope_theta_local=10000.0)
DESCS["tiny_modern"] = dict(layers=4, hidden=128, heads=2, ffn=192, vocab=8192, num_labels=9, max_pos=512, ln_eps=1e-5,
                            dtype=0, **_MODERN)
DESCS["base_modern"] = dict(layers=22, hidden=768, heads=12, ffn=1152, vocab=50368, num_labels=13, max_pos=512, ln_eps=1e-5,
                            dtype=1, **_MODERN)
TYPE_NAMES_6 = ["IP_ADDRESS", "IPV6_ADDRESS", "HOSTNAME", "CVE_ID", "MAC_ADDRESS", "SERIAL_NUMBER"]
TYPE_NAMES_4 = ["TYPE0", "TYPE1", "TYPE2", "TYPE3"]
# rule D17's pattern set: one pattern per synthetic entity kind of entity_pool(), in type order (data for the NEXT-4
# regex layer: the patterns are inputs of the method, like the key and the type names)
REGEX_PATTERNS = [r"(?:[0-9]{1,3}\.){3}[0-9]{1,3}", r"(?:[0-9a-f]{1,4}:){7}[0-9a-f]{1,4}",
                  r"(?:[a-z0-9]+\.)+(?:example|internal|corp|lan|test|invalid)", r"CVE-[0-9]{4}-[0-9]{4,7}",
                  r"(?:[0-9a-f]{2}:){5}[0-9a-f]{2}", r"[0-9a-f]{16,32}"]
PAD, CLS, SEP, UNK, MASK = 0, 1, 2, 3, 4
# W2 planted-detector strengths: (alpha, beta, gamma) plants the embedding bands and the
# head only; the 6-tuple adds (kappa, theta, lam), one re-amplifying FFN unit per class in every layer (make_weights), which a
# 24-layer stack needs -- with the 3-tuple the oracle itself labels no entity token at L = 24 and only 79 % of them at L = 12.
PLANTED = (2.0, 0.5, 4.0)
PLANTED_DEEP = (2.0, 0.5, 4.0, 1.0, 8.0, 1.0)
FIRST_ID = 5
BAND = 256


def rng(seed):
    return np.random.Generator(np.random.PCG64(seed))


def bf16_round(a):
    """Round fp32 values to the nearest BF16 (ties to even), returned as fp32 (W0)."""
    u = np.ascontiguousarray(a, np.float32).view(np.uint32).astype(np.uint64)
    u = (u + 0x7FFF + ((u >> 16) & 1)) & 0xFFFF0000
    return u.astype(np.uint32).view(np.float32).reshape(np.shape(a))


LAYER_ORDER = ["W_qkv", "b_qkv", "W_o", "b_o", "g_1", "b_1", "W_1", "b_1f", "W_2", "b_2f", "g_2", "b_2"]
MATRICES = {"E_w", "E_p", "W_qkv", "W_o", "W_1", "W_2", "W_c"}   # rounded to BF16 when dtype=1


def make_weights(desc, seed, planted=None):
    """W1 (pure N(0,0.02)) or W2 (planted detector: planted=(alpha, beta, gamma)) parameters.

    Returns a dict of fp32 arrays (names of SURVEY §8(c) O1) with key "layers" = list of dicts.
    For dtype=1 every matrix/embedding is rounded to BF16 so both sides consume identical values.
    """
    g = rng(seed)
    H, F, V, NL, P, L = (desc[k] for k in ("hidden", "ffn", "vocab", "num_labels", "max_pos", "layers"))
    n = lambda *s: (0.02 * g.standard_normal(s)).astype(np.float32)
    gam = lambda: (1.0 + 0.02 * g.standard_normal(H)).astype(np.float32)
    w = {"E_w": n(V, H), "E_p": n(P, H), "E_t": n(H), "g_e": gam(), "b_e": n(H), "layers": []}
    for _ in range(L):
        w["layers"].append({
            "W_qkv": n(3 * H, H), "b_qkv": n(3 * H), "W_o": n(H, H), "b_o": n(H), "g_1": gam(), "b_1": n(H),
            "W_1": n(F, H), "b_1f": n(F), "W_2": n(H, F), "b_2f": n(H), "g_2": gam(), "b_2": n(H)})
    w["W_c"] = n(NL, H)
    w["b_c"] = n(NL)
    if planted is not None:
        alpha, beta, gamma = planted[:3]
        q, _ = np.linalg.qr(g.standard_normal((H, NL - 1)))
        for c in range(1, NL):
            u = q[:, c - 1].astype(np.float32)
            lo = FIRST_ID + (c - 1) * BAND
            w["E_w"][lo:lo + BAND] += alpha * u
            w["W_c"][c] += beta * u
        w["b_c"][0] += gamma
        if len(planted) == 6:
            # W2 "deep" variant: every layer also carries one FFN unit per class that re-amplifies the planted direction when
            # it is clearly present (unit c-1: pre-activation kappa * (x . u_c) - theta, output lam * u_c), so that the detector
            # survives the LayerNorm rescaling of a deep stack (24 layers fade the embedding-only plant to nothing)
            kappa, theta, lam = planted[3:]
            for lw in w["layers"]:
                for c in range(1, NL):
                    u = q[:, c - 1].astype(np.float32)
                    lw["W_1"][c - 1] += kappa * u
                    lw["b_1f"][c - 1] -= theta
                    lw["W_2"][:, c - 1] += lam * u
    if desc["dtype"] == 1:
        for k in ("E_w", "E_p", "W_c"):
            w[k] = bf16_round(w[k])
        for lw in w["layers"]:
            for k in ("W_qkv", "W_o", "W_1", "W_2"):
                lw[k] = bf16_round(lw[k])
    return w


MODERN_LAYER_ORDER = ["g_a", "W_qkv", "W_o", "g_m", "W_i", "W_2"]


def make_weights_modern(desc, seed, planted=None):
    """Parameters of the arch-1 encoder (names of oracle/encoder_modern.py); W1 or planted-detector W2 like make_weights."""
    g = rng(seed)
    H, F, V, NL, L = (desc[k] for k in ("hidden", "ffn", "vocab", "num_labels", "layers"))
    n = lambda *s: (0.02 * g.standard_normal(s)).astype(np.float32)
    gam = lambda: (1.0 + 0.02 * g.standard_normal(H)).astype(np.float32)
    w = {"E_w": n(V, H), "g_e": gam(), "layers": []}
    for _ in range(L):
        w["layers"].append({"g_a": gam(), "W_qkv": n(3 * H, H), "W_o": n(H, H), "g_m": gam(), "W_i": n(2 * F, H), "W_2": n(H, F)})
    w["g_f"] = gam()
    w["W_c"] = n(NL, H)
    w["b_c"] = n(NL)
    if planted is not None:
        alpha, beta, gamma = planted
        q, _ = np.linalg.qr(g.standard_normal((H, NL - 1)))
        for c in range(1, NL):
            u = q[:, c - 1].astype(np.float32)
            lo = FIRST_ID + (c - 1) * BAND
            w["E_w"][lo:lo + BAND] += alpha * u
            w["W_c"][c] += beta * u
        w["b_c"][0] += gamma
    if desc["dtype"] == 1:
        for k in ("E_w", "W_c"):
            w[k] = bf16_round(w[k])
        for lw in w["layers"]:
            for k in ("W_qkv", "W_o", "W_i", "W_2"):
                lw[k] = bf16_round(lw[k])
    return w


def pack_blob_modern(w):
    """Flat fp32 blob of the arch-1 parameters in the ABI's order: E_w, g_e, {g_a, W_qkv, W_o, g_m, W_i, W_2} x L, g_f, W_c, b_c."""
    parts = [w["E_w"], w["g_e"]]
    for lw in w["layers"]:
        parts += [lw[k] for k in MODERN_LAYER_ORDER]
    parts += [w["g_f"], w["W_c"], w["b_c"]]
    return np.concatenate([np.ascontiguousarray(p, np.float32).ravel() for p in parts])


def pack_blob(w):
    """Flat fp32 blob in the ABI's fixed order (include/anonshield.h, anon_weights_load)."""
    parts = [w[k] for k in ("E_w", "E_p", "E_t", "g_e", "b_e")]
    for lw in w["layers"]:
        parts += [lw[k] for k in LAYER_ORDER]
    parts += [w["W_c"], w["b_c"]]
    return np.concatenate([np.ascontiguousarray(p, np.float32).ravel() for p in parts])


# ---- config 1: padded + packed token ids -----------------------------------------------------
def tokens_uniform(n_seqs, len_lo, len_hi, vocab, seed, max_len=None):
    """Lengths U{len_lo..len_hi}, ids U[5, vocab).  Returns (ids, cu_seqlens, ids_padded, lengths)."""
    g = rng(seed)
    lengths = g.integers(len_lo, len_hi + 1, n_seqs).astype(np.int32)
    cu = np.zeros(n_seqs + 1, np.int32)
    cu[1:] = np.cumsum(lengths)
    ids = g.integers(FIRST_ID, vocab, int(cu[-1])).astype(np.int32)
    Lmax = max_len or int(lengths.max())
    padded = np.full((n_seqs, Lmax), PAD, np.int32)
    for i in range(n_seqs):
        padded[i, :lengths[i]] = ids[cu[i]:cu[i + 1]]
    return ids, cu, padded, lengths


# ---- entity-string pools and span lists ----------------------------------------------------------
def ascii_pool(n_unique, len_lo, len_hi, seed):
    """n_unique distinct printable-ASCII (0x21-0x7E) strings, lengths U{len_lo..len_hi}: CSR."""
    g = rng(seed)
    lens = g.integers(len_lo, len_hi + 1, n_unique).astype(np.int64)
    off = np.zeros(n_unique + 1, np.int64)
    off[1:] = np.cumsum(lens)
    data = g.integers(0x21, 0x7F, int(off[-1])).astype(np.uint8)
    # make them distinct by construction: overwrite the first bytes with a base-94 index
    idx = np.arange(n_unique, dtype=np.int64)
    ndig = 1
    while 94 ** ndig < n_unique:
        ndig += 1
    assert ndig <= len_lo, "pool too large for the minimum length"
    for d in range(ndig):
        data[off[:-1] + d] = (0x21 + (idx // (94 ** d)) % 94).astype(np.uint8)
    return data, off


def zipf_draws(n_unique, n_draws, s, seed):
    """Ranks 0..n_unique-1 drawn with P(k) ~ (k+1)^-s by inverse CDF; rank -> string by a seeded shuffle."""
    g = rng(seed)
    wts = np.arange(1, n_unique + 1, dtype=np.float64) ** (-s)
    cdf = np.cumsum(wts)
    cdf /= cdf[-1]
    r = np.searchsorted(cdf, g.random(n_draws), side="left")
    np.minimum(r, n_unique - 1, out=r)
    perm = g.permutation(n_unique)
    return perm[r].astype(np.int64)


def expand_csr(pool, pool_off, draws, chunk=1 << 20):
    """span list CSR (bytes, int64 offsets) = pool strings in the order of draws (pure gather)."""
    lens = (pool_off[1:] - pool_off[:-1])[draws]
    off = np.zeros(len(draws) + 1, np.int64)
    off[1:] = np.cumsum(lens)
    out = np.empty(int(off[-1]), np.uint8)
    for a in range(0, len(draws), chunk):
        b = min(a + chunk, len(draws))
        ln = lens[a:b]
        src0 = pool_off[draws[a:b]]
        dst = off[a]
        total = int(off[b] - off[a])
        within = np.arange(total, dtype=np.int64) - np.repeat(off[a:b] - dst, ln)
        out[dst:dst + total] = pool[np.repeat(src0, ln) + within]
    return out, off


def spans_config1(seed=SEED_BASE + 1):
    """700 unique ASCII strings of 4-64 bytes + 300 re-draws, shuffled; types U{0..3}; 32-byte key."""
    g = rng(seed)
    pool, poff = ascii_pool(700, 4, 64, seed + 1000)
    draws = np.concatenate([np.arange(700), g.integers(0, 700, 300)])
    g.shuffle(draws)
    data, off = expand_csr(pool, poff, draws)
    types = g.integers(0, 4, 1000).astype(np.uint8)
    key = g.integers(0, 256, 32).astype(np.uint8)
    return data, off, types, key


def spans_zipf(n_unique, n_draws, len_lo, len_hi, n_types, seed, s=1.1):
    """Config 5 shape: Zipf(s) draws over a pool of printable-ASCII strings (CSR), types, key."""
    g = rng(seed)
    pool, poff = ascii_pool(n_unique, len_lo, len_hi, seed + 1000)
    draws = zipf_draws(n_unique, n_draws, s, seed + 2000)
    data, off = expand_csr(pool, poff, draws)
    types = g.integers(0, n_types, n_draws).astype(np.uint8)
    key = g.integers(0, 256, 32).astype(np.uint8)
    return data, off, types, key, draws


# ---- synthetic records, tokenizer and windowing (host glue outside the hot path) ------------------
def _hexs(vals, width):
    return [format(int(v), "0%dx" % width) for v in vals]


def entity_pool(n_unique, seed):
    """n_unique distinct entity strings of 6 kinds (IPv4, IPv6, host name, CVE-shaped, MAC, hex serial).

    Returns (bytes, int64 offsets, uint8 type).  Distinct by construction (an index is folded in)."""
    g = rng(seed)
    kinds = g.integers(0, 6, n_unique)
    strs = []
    syl = ["srv", "db", "web", "mail", "gw", "app", "node", "edge", "core", "vpn", "lab", "dev", "ops", "net"]
    tld = ["example", "internal", "corp", "lan", "test", "invalid"]
    counters = [0] * 6
    for i in range(n_unique):
        k = int(kinds[i])
        c = counters[k]
        counters[k] += 1
        if k == 0:
            v = (c * 2654435761 + 0x0A000001) & 0xFFFFFFFF
            s = "%d.%d.%d.%d" % (v >> 24, (v >> 16) & 255, (v >> 8) & 255, v & 255)
        elif k == 1:
            hi = int(g.integers(0, 1 << 62))
            groups = [0x2001, 0x0DB8, (hi >> 32) & 0xFFFF, (hi >> 16) & 0xFFFF, hi & 0xFFFF,
                      (c >> 32) & 0xFFFF, (c >> 16) & 0xFFFF, c & 0xFFFF]
            if c % 3 == 0:   # compressed form: drop one zero group run if present
                s = ":".join("%x" % x for x in groups)
            else:
                s = ":".join("%04x" % x for x in groups)
        elif k == 2:
            nlab = 2 + c % 3
            labs = ["%s%d" % (syl[(c // 7 + j) % len(syl)], c if j == 0 else (c >> (3 * j)) % 10) for j in range(nlab - 1)]
            s = ".".join(labs + [tld[c % len(tld)]])
        elif k == 3:
            s = "CVE-%d-%d" % (1999 + c % 27, 1000 + c // 27)
        elif k == 4:
            v = (c * 0x9E3779B97F4A7C15 + 0x020000000000) & 0xFFFFFFFFFFFF
            s = ":".join("%02x" % ((v >> (8 * j)) & 255) for j in range(5, -1, -1))
        else:
            width = 16 + 2 * (c % 9)                       # 16..32 hex chars
            s = format((c * 0x9E3779B97F4A7C15 + (1 << 63)) & ((1 << 64) - 1), "016x")
            if width > 16:
                s += format(c % (16 ** (width - 16)), "x").zfill(width - 16)
        strs.append(s.encode())
    assert len(set(strs)) == n_unique, "entity pool not distinct"
    lens = np.fromiter((len(s) for s in strs), np.int64, n_unique)
    off = np.zeros(n_unique + 1, np.int64)
    off[1:] = np.cumsum(lens)
    data = np.frombuffer(b"".join(strs), np.uint8).copy()
    return data, off, kinds.astype(np.uint8)


def _filler_pool(n_words, seed):
    g = rng(seed)
    lens = g.integers(1, 7, n_words).astype(np.int64)
    mat = g.integers(ord("a"), ord("z") + 1, (n_words, 6)).astype(np.uint8)
    return lens, mat


def _piece_hash(mat, lens):
    """Band index of an entity piece = simple polynomial hash of its <=4 bytes mod 256."""
    h = np.zeros(mat.shape[0], np.int64)
    for j in range(mat.shape[1]):
        h = np.where(j < lens, (h * 131 + mat[:, j]) & 0xFFFFFFFF, h)
    return (h ^ (h >> 9)) % BAND


def make_records(n_records, content_tokens, desc, pool, pool_off, pool_type, seed, zipf_s=None,
                 entity_rate=1.0 / 25):
    """Synthetic record stream + its tokenisation (SURVEY §8(d) "Synthetic tokenizer").

    content_tokens[r] = number of content tokens of record r.  Words are joined by single
    spaces; an entity string is cut into pieces of <= 4 bytes that are adjacent in the text;
    first piece id in the B-t band, later pieces in the I-t band; filler word ids follow the
    bands.  One entity after every Geometric(entity_rate) filler tokens.

    Returns dict(text uint8[], rec_off int64[R+1], tok_rec_off int64[R+1], ids int32[N],
    char_start int32[N], char_end int32[N], planted_label int8[N], ent_draws list).
    """
    g = rng(seed)
    NL = desc["num_labels"]
    filler_base = FIRST_ID + (NL - 1) * BAND
    n_filler = desc["vocab"] - filler_base
    flen, fmat = _filler_pool(n_filler, seed + 77)
    n_pool = len(pool_off) - 1
    plen_all = pool_off[1:] - pool_off[:-1]
    if zipf_s is not None:
        wts = np.arange(1, n_pool + 1, dtype=np.float64) ** (-zipf_s)
        cdf = np.cumsum(wts)
        cdf /= cdf[-1]
        perm = g.permutation(n_pool)
    texts, ids_l, cs_l, ce_l, lab_l = [], [], [], [], []
    rec_off = np.zeros(n_records + 1, np.int64)
    tok_off = np.zeros(n_records + 1, np.int64)
    n_ent_total = 0
    for r in range(n_records):
        n = int(content_tokens[r])
        kmax = max(4, int(n * entity_rate * 2) + 4)
        gaps = g.geometric(entity_rate, kmax)                  # >= 1 filler before each entity
        if zipf_s is not None:
            ent = perm[np.minimum(np.searchsorted(cdf, g.random(kmax)), n_pool - 1)]
        else:
            ent = g.integers(0, n_pool, kmax)
        elen = plen_all[ent]
        pieces = (elen + 3) // 4
        end_tok = np.cumsum(gaps + pieces)
        k = int(np.searchsorted(end_tok, n, side="right"))     # entities that fit entirely
        gaps, ent, elen, pieces = gaps[:k], ent[:k], elen[:k], pieces[:k]
        n_ent_total += k
        # token-level layout
        is_ent = np.zeros(n, bool)
        first_piece = np.zeros(n, bool)
        tok_ent = np.full(n, -1, np.int64)      # which entity (0..k-1) a piece belongs to
        tok_piece = np.zeros(n, np.int64)
        if k:
            start = np.cumsum(gaps + pieces) - pieces          # first token index of each entity
            tot = int(pieces.sum())
            within = np.arange(tot) - np.repeat(np.cumsum(pieces) - pieces, pieces)
            pos = np.repeat(start, pieces) + within
            is_ent[pos] = True
            tok_ent[pos] = np.repeat(np.arange(k), pieces)
            tok_piece[pos] = within
            first_piece[start] = True
        # byte length of every token
        fw = g.integers(0, n_filler, n)
        tlen = flen[fw].copy()
        if k:
            e_of = tok_ent[is_ent]
            tlen[is_ent] = np.minimum(4, elen[e_of] - 4 * tok_piece[is_ent])
        sep = np.ones(n, np.int64)               # one space before every unit except the first token
        sep[is_ent & ~first_piece] = 0
        sep[0] = 0
        cstart = np.cumsum(sep + tlen) - tlen
        cend = cstart + tlen
        nbytes = int(cend[-1]) if n else 0
        text = np.full(nbytes, ord(" "), np.uint8)
        # token bytes: [n, 6] matrix, then masked scatter
        tb = fmat[fw]
        if k:
            src = pool_off[ent][e_of] + 4 * tok_piece[is_ent]
            eb = np.zeros((len(src), 6), np.uint8)
            for j in range(4):
                ok = j < tlen[is_ent]
                eb[ok, j] = pool[src[ok] + j]
            tb = tb.copy()
            tb[is_ent] = eb
        col = np.arange(6)[None, :]
        mask = col < tlen[:, None]
        text[(cstart[:, None] + col)[mask]] = tb[mask]
        # ids and planted labels
        ids = (filler_base + fw).astype(np.int32)
        lab = np.zeros(n, np.int8)
        if k:
            t_of = pool_type[ent][e_of].astype(np.int64)
            cls = np.where(tok_piece[is_ent] == 0, 2 * t_of + 1, 2 * t_of + 2)
            hidx = _piece_hash(tb[is_ent][:, :4], tlen[is_ent])
            ids[is_ent] = (FIRST_ID + (cls - 1) * BAND + hidx).astype(np.int32)
            lab[is_ent] = cls
        texts.append(text)
        ids_l.append(ids)
        cs_l.append(cstart.astype(np.int32))
        ce_l.append(cend.astype(np.int32))
        lab_l.append(lab)
        rec_off[r + 1] = rec_off[r] + nbytes
        tok_off[r + 1] = tok_off[r] + n
    cat = lambda l, dt: np.concatenate(l) if l else np.zeros(0, dt)
    return dict(text=cat(texts, np.uint8), rec_off=rec_off, tok_rec_off=tok_off, ids=cat(ids_l, np.int32),
                char_start=cat(cs_l, np.int32), char_end=cat(ce_l, np.int32),
                planted_label=cat(lab_l, np.int8), n_entities=n_ent_total)


def field_spans(rec, fixed_type):
    """NEXT-2 input (PAPER.md L57 `anonymization_config`): the caller-supplied FIELD spans of a record stream -- the byte range
    of every generated entity string, all with one fixed type -- as int32 [S, 4] rows (record, char_start, char_end, type) in
    stream order.  Pure layout: the ranges are where make_records put the strings (a run of labelled pieces; every entity is
    preceded by at least one filler token, so runs never touch or cross a record)."""
    lab = rec["planted_label"]
    n = lab.size
    starts = np.flatnonzero((lab > 0) & (lab % 2 == 1))
    zeros = np.flatnonzero(lab == 0)
    nxt = np.searchsorted(zeros, starts)                       # first unlabelled token after each start
    ends = np.where(nxt < zeros.size, zeros[np.minimum(nxt, zeros.size - 1)], n) - 1
    tok_rec = np.searchsorted(rec["tok_rec_off"], starts, side="right") - 1
    out = np.empty((starts.size, 4), np.int32)
    out[:, 0] = tok_rec
    out[:, 1] = rec["char_start"][starts]
    out[:, 2] = rec["char_end"][ends]
    out[:, 3] = fixed_type
    return out


WINDOW_CONTENT, WINDOW_OVERLAP = 510, 128
WINDOW_STRIDE = WINDOW_CONTENT - WINDOW_OVERLAP


def window_records(rec, rec_subset=None):
    """Cut every record into 510+2-token windows with 128-token overlap and midpoint ownership.

    Returns dict(token_ids int32[T], cu_seqlens int32[B+1], meta int32[T,4], win_rec int32[B],
    planted_label int8[T]) -- the hot path's inputs."""
    tok_off = rec["tok_rec_off"]
    recs = range(len(tok_off) - 1) if rec_subset is None else rec_subset
    ids_l, meta_l, lab_l, lens, wrec = [], [], [], [], []
    for r in recs:
        a, n = int(tok_off[r]), int(tok_off[r + 1] - tok_off[r])
        W = 1 if n <= WINDOW_CONTENT else 1 + -(-(n - WINDOW_CONTENT) // WINDOW_STRIDE)
        for w in range(W):
            lo = WINDOW_STRIDE * w
            hi = min(lo + WINDOW_CONTENT, n)
            gidx = np.arange(lo, hi)
            keep = np.ones(hi - lo, bool)
            if w + 1 < W:
                keep &= gidx < WINDOW_STRIDE * (w + 1) + WINDOW_OVERLAP // 2
            if w > 0:
                keep &= gidx >= WINDOW_STRIDE * w + WINDOW_OVERLAP // 2
            m = np.zeros((hi - lo + 2, 4), np.int32)
            m[:, 0] = r
            m[1:-1, 1] = rec["char_start"][a + lo:a + hi]
            m[1:-1, 2] = rec["char_end"][a + lo:a + hi]
            m[1:-1, 3] = keep
            ids = np.empty(hi - lo + 2, np.int32)
            ids[0], ids[-1] = CLS, SEP
            ids[1:-1] = rec["ids"][a + lo:a + hi]
            lab = np.zeros(hi - lo + 2, np.int8)
            lab[1:-1] = rec["planted_label"][a + lo:a + hi]
            ids_l.append(ids)
            meta_l.append(m)
            lab_l.append(lab)
            lens.append(hi - lo + 2)
            wrec.append(r)
    cu = np.zeros(len(lens) + 1, np.int32)
    cu[1:] = np.cumsum(lens)
    return dict(token_ids=np.concatenate(ids_l), cu_seqlens=cu, meta=np.concatenate(meta_l),
                win_rec=np.asarray(wrec, np.int32), planted_label=np.concatenate(lab_l))


def lognormal_lengths(n, median, sigma, lo, hi, seed):
    g = rng(seed)
    return np.clip(np.round(g.lognormal(np.log(median), sigma, n)), lo, hi).astype(np.int64)


# ---- the named workloads ----------------------------------------------------------------------------
def workload_base(n_records=4096, seed=SEED_BASE + 2, n_pool=50000, desc=None):
    """Config 2: one sequence per record, content length clip(round(LogNormal(ln 200, 0.75)), 8, 510)."""
    desc = desc or DESCS["base"]
    pool, poff, ptype = entity_pool(n_pool, seed + 1)
    n_tok = lognormal_lengths(n_records, 200, 0.75, 8, 510, seed + 2)
    rec = make_records(n_records, n_tok, desc, pool, poff, ptype, seed + 3)
    win = window_records(rec)
    return rec, win


def workload_stream(n_records=70951, seed=SEED_BASE + 3, n_pool=300000, desc=None):
    """Config 3: record bytes = min(LogNormal(ln 4096, 1.168), 65536) at ~4 B/token; Zipf(1.1) entities."""
    desc = desc or DESCS["base"]
    pool, poff, ptype = entity_pool(n_pool, seed + 1)
    g = rng(seed + 2)
    nbytes = np.minimum(g.lognormal(np.log(4096), 1.168, n_records), 65536.0)
    n_tok = np.maximum(np.round(nbytes / 4.0), 8).astype(np.int64)
    rec = make_records(n_records, n_tok, desc, pool, poff, ptype, seed + 3, zipf_s=1.1)
    return rec


def workload_large(n_seqs=16384, seed=SEED_BASE + 4, n_pool=50000, desc=None):
    """Config 4: total length U{32..512} including the two specials."""
    desc = desc or DESCS["large"]
    pool, poff, ptype = entity_pool(n_pool, seed + 1)
    n_tok = rng(seed + 2).integers(30, 511, n_seqs).astype(np.int64)
    rec = make_records(n_seqs, n_tok, desc, pool, poff, ptype, seed + 3)
    win = window_records(rec)
    return rec, win
