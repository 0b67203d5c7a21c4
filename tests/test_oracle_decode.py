"""Pins for oracle/decode.py (BIO decode, window stitch, gather) -- CPU only."""
import itertools
import os

import numpy as np

from oracle import decode

CHARS = [(0, 3), (4, 7), (8, 11), (12, 15), (16, 19), (20, 23)]


def _parse_case(line):
    lab_s, span_s = [x.strip() for x in line.split(";")]
    labels, meta, rec, pos = [], [], 0, 0
    for tok in lab_s.split():
        if tok == "|":
            rec, pos = rec + 1, 0
            continue
        keep = 1
        if tok.startswith("k"):
            keep, tok = 0, tok[1:]
        labels.append(int(tok))
        meta.append((rec, CHARS[pos][0], CHARS[pos][1], keep))
        pos += 1
    spans = [] if span_s == "-" else [tuple(int(v) for v in s.split(":")) for s in span_s.split()]
    return np.array(labels), np.array(meta), spans


def test_hand_worked_bio_cases(golden_dir):
    n = 0
    with open(os.path.join(golden_dir, "bio_cases.txt")) as f:
        for line in f:
            if not line.strip() or line.startswith("#"):
                continue
            labels, meta, want = _parse_case(line)
            assert decode.decode_spans(labels, meta) == want, line
            n += 1
    assert n == 10


def _rederive(labels, meta):
    """Independent restatement of the three bullet rules of SURVEY §8(c) O3 via start/continue flags."""
    kept = [j for j in range(len(labels)) if meta[j][3] & 1]
    starts, conts = [], []
    for idx, j in enumerate(kept):
        lab = labels[j]
        p = kept[idx - 1] if idx > 0 and meta[kept[idx - 1]][0] == meta[j][0] else None
        cont = lab > 0 and lab % 2 == 0 and p is not None and labels[p] > 0 and (labels[p] - 1) // 2 == (lab - 1) // 2
        conts.append(cont)
        starts.append(lab > 0 and not cont)
    spans = []
    for idx, j in enumerate(kept):
        if starts[idx]:
            e = idx
            while e + 1 < len(kept) and conts[e + 1]:
                e += 1
            spans.append((int(meta[j][0]), int(meta[j][1]), int(meta[kept[e]][2]), int((labels[j] - 1) // 2)))
    return spans


def test_exhaustive_nt1_and_random_nt3():
    # exhaustive for NT = 1 (labels 0..2), T = 7, with a record break after token 3 and one non-kept token
    for T in (1, 4, 7):
        for labs in itertools.product(range(3), repeat=T):
            meta = np.array([(0 if j < 3 else 1, 5 * j, 5 * j + 4, 0 if j == 2 else 1) for j in range(T)])
            assert decode.decode_spans(np.array(labs), meta) == _rederive(np.array(labs), meta)
    g = np.random.default_rng(3)
    for _ in range(300):
        T = int(g.integers(0, 13))
        labs = g.integers(0, 7, T)
        rec = np.cumsum(g.random(T) < 0.15)
        meta = np.stack([rec, 4 * np.arange(T), 4 * np.arange(T) + 3, (g.random(T) < 0.8).astype(int)], 1) if T else np.zeros((0, 4), int)
        assert decode.decode_spans(labs, meta) == _rederive(labs, meta)


def test_window_plan_every_token_kept_exactly_once():
    for n in [1, 8, 509, 510, 511, 638, 639, 892, 893, 1274, 1275, 5000, 16384]:
        plan = decode.window_plan(n)
        assert len(plan) == decode.num_windows(n)
        count = np.zeros(n, int)
        for w, (lo, hi, keep) in enumerate(plan):
            assert lo == 382 * w and hi == min(lo + 510, n) and hi - lo == len(keep)
            count[lo:hi] += np.array(keep, int)
            if w + 1 < len(plan):           # overlap with the next window is exactly 128 tokens
                assert hi - 382 * (w + 1) == 128
        assert (count == 1).all(), n
        # each kept token has >= 64 tokens of context on a cut side
        for w, (lo, hi, keep) in enumerate(plan):
            ks = [lo + i for i, k in enumerate(keep) if k]
            if w > 0:
                assert min(ks) - lo >= 64
            if w + 1 < len(plan):
                assert hi - 1 - max(ks) >= 64


def test_stitched_decode_independent_of_window_boundaries():
    """Labels supplied directly: decoding the windowed stream == decoding the un-windowed record."""
    g = np.random.default_rng(5)
    for n in [700, 1300]:
        labs = g.integers(0, 5, n) * (g.random(n) < 0.5)
        cs = 5 * np.arange(n)
        flat_meta = np.stack([np.zeros(n, int), cs, cs + 4, np.ones(n, int)], 1)
        want = decode.decode_spans(labs, flat_meta)
        wl, wm = [], []
        for lo, hi, keep in decode.window_plan(n):
            wl += [9] + list(labs[lo:hi]) + [9]       # specials carry a junk label: never read (keep = 0)
            wm += [(0, 0, 0, 0)] + [(0, cs[t], cs[t] + 4, int(k)) for t, k in zip(range(lo, hi), keep)] + [(0, 0, 0, 0)]
        assert decode.decode_spans(np.array(wl), np.array(wm)) == want


def test_gather_spans():
    text = np.frombuffer(b"hello world" + b"abc 10.0.0.1 xyz", np.uint8)
    rec_off = np.array([0, 11, 27])
    data, off = decode.gather_spans(text, rec_off, [(0, 6, 11, 0), (1, 4, 12, 1), (1, 0, 0, 0)])
    assert bytes(data) == b"world10.0.0.1" and off.tolist() == [0, 5, 13, 13]


def test_splice_records_hand_worked_and_library_replace():
    """NEXT-1 pins: a hand-worked record pair; str.replace on records whose entity strings occur exactly once (an
    independent library routine); zero spans = identity; total length = original + sum of (token - span) lengths;
    splicing the originals back in place of the tokens recovers the input."""
    text = np.frombuffer(b"ip 10.0.0.1 seen" + b"host a.b and 10.0.0.1", np.uint8)
    rec_off = np.array([0, 16, 37], np.int64)
    spans = [(0, 3, 11, 0), (1, 5, 8, 2), (1, 13, 21, 0)]
    toks = [b"[IP_ADDRESS_aaaaaaaaaa]", b"[HOSTNAME_bbbbbbbbbb]", b"[IP_ADDRESS_aaaaaaaaaa]"]
    tok = np.frombuffer(b"".join(toks), np.uint8)
    toff = np.array([0] + list(np.cumsum([len(t) for t in toks])), np.int64)
    out, ooff = decode.splice_records(text, rec_off, spans, tok, toff)
    assert bytes(out[ooff[0]:ooff[1]]) == b"ip [IP_ADDRESS_aaaaaaaaaa] seen"
    assert bytes(out[ooff[1]:ooff[2]]) == b"host [HOSTNAME_bbbbbbbbbb] and [IP_ADDRESS_aaaaaaaaaa]"
    # identity with no spans
    o2, f2 = decode.splice_records(text, rec_off, [], np.zeros(0, np.uint8), np.zeros(1, np.int64))
    assert np.array_equal(o2, text) and np.array_equal(f2, rec_off)
    # seeded records with unique entity strings: sequential str.replace gives the same bytes
    rng = np.random.default_rng(4)
    recs, sp, tk = [], [], []
    for r in range(20):
        words, pos, body = [], 0, b""
        for k in range(int(rng.integers(0, 7))):
            filler = bytes(rng.integers(97, 123, int(rng.integers(0, 9))).astype(np.uint8))
            ent = b"<E%d_%d>" % (r, k)
            body += filler + b" "
            sp.append((r, len(body), len(body) + len(ent), k % 3))
            tk.append(b"[T%d_%04x]" % (k % 3, int(rng.integers(0, 65536))) if k % 2 else b"[]")   # longer and shorter than the span
            body += ent + b" "
        recs.append(body + bytes(rng.integers(97, 123, int(rng.integers(0, 5))).astype(np.uint8)))
    text2 = np.frombuffer(b"".join(recs), np.uint8)
    roff = np.array([0] + list(np.cumsum([len(b) for b in recs])), np.int64)
    tok2 = np.frombuffer(b"".join(tk), np.uint8)
    toff2 = np.array([0] + list(np.cumsum([len(t) for t in tk])), np.int64)
    out3, ooff3 = decode.splice_records(text2, roff, sp, tok2, toff2)
    for r in range(20):
        want = recs[r]
        for (rr, cs, ce, _t), t in zip(sp, tk):
            if rr == r:
                want = want.replace(recs[r][cs:ce], t)
        assert bytes(out3[ooff3[r]:ooff3[r + 1]]) == want
    assert out3.size == text2.size + sum(len(t) - (ce - cs) for (_r, cs, ce, _t), t in zip(sp, tk))
    # inverse splice: put the original strings back where the tokens now are
    inv_spans, shift, last = [], 0, -1
    for (r, cs, ce, t), tkn in zip(sp, tk):
        if r != last:
            shift, last = 0, r
        inv_spans.append((r, cs + shift, cs + shift + len(tkn), t))
        shift += len(tkn) - (ce - cs)
    ent_bytes, ent_off = decode.gather_spans(text2, roff, sp)
    back, boff = decode.splice_records(out3, ooff3, inv_spans, ent_bytes, ent_off)
    assert np.array_equal(back, text2) and np.array_equal(boff, roff)
