"""GPU parity of NEXT-4: the DFA regex scan and the regex / NER span merge against
oracle/regex_layer.py, bit-exact, through the C ABI; then the whole host pipeline with an attached automaton against
the oracle composition encoder -> decode -> merge -> gather -> pseudonymize -> splice."""
import numpy as np
import pytest

from harness import gen

pytestmark = pytest.mark.gpu


def _env():
    import torch
    import paper_2606_15650_b200 as P
    if not torch.cuda.is_available():
        pytest.fail("GPU test selected but no CUDA device")
    return torch, P


def _blob(max_match=None):
    from oracle import regex_layer as rx
    from paper_2606_15650_b200 import regex_dfa
    return regex_dfa.compile_patterns([(k, p) for k, (_n, p) in enumerate(rx.PATTERNS)], max_match or rx.MAX_MATCH)


def _scan_gpu(torch, P, ctx, R, text, rec_off, cap):
    dev = torch.device("cuda", 0)
    d_text = torch.from_numpy(np.ascontiguousarray(text)).to(dev)
    d_off = torch.from_numpy(np.ascontiguousarray(rec_off, np.int64)).to(dev)
    spans = torch.full((max(cap, 1), 4), -7, dtype=torch.int32, device=dev)[:cap]
    num = torch.full((1,), -1, dtype=torch.int32, device=dev)
    P.anon_regex_scan(ctx, R, d_text, d_off, spans, num)
    rc = ctx.sync()
    n = int(num.item())
    return rc, n, spans[:min(n, cap)].cpu().numpy()


def _records(n_records, seed, median=300):
    d = dict(gen.DESCS["tiny"])
    pool, poff, ptype = gen.entity_pool(400, seed)
    g = gen.rng(seed + 1)
    n_tok = np.minimum(g.lognormal(np.log(median), 1.0, n_records), 6000).astype(np.int64) + 8
    return d, gen.make_records(n_records, n_tok, d, pool, poff, ptype % 4, seed + 2, zipf_s=1.1, entity_rate=1.0 / 12), (pool, poff, ptype)


def test_regex_scan_matches_oracle_on_record_stream():
    from oracle import regex_layer as rx
    torch, P = _env()
    d, rec, _pool = _records(160, 31)
    text, off = rec["text"], rec["rec_off"]
    assert text.size > 5 * 4096                                            # several tiles and a ragged tail
    want = rx.scan_records(text, off)
    assert len(want) > 500 and len({s[3] for s in want}) == 6              # every pattern kind occurs
    ctx = P.Context(0, workspace_bytes=64 << 20)
    R = P.Regex(ctx, _blob())
    rc, n, got = _scan_gpu(torch, P, ctx, R, text, off, len(want) + 10)
    assert rc == 0 and n == len(want)
    assert np.array_equal(got, np.asarray(want, np.int32).reshape(-1, 4))
    # capacity: the total is still reported, the prefix is written, CAPACITY is latched
    rc, n, got = _scan_gpu(torch, P, ctx, R, text, off, 100)
    assert rc == P.binding.ERR_CAPACITY and n == len(want)
    assert np.array_equal(got, np.asarray(want[:100], np.int32).reshape(-1, 4))
    R.close(); ctx.close()


def test_regex_scan_dense_candidates_and_degenerate_records():
    """Random text over a small alphabet (candidates at most positions, overlapping candidates, matches cut by record
    boundaries and by max_match), empty records, one-byte records, a record longer than several tiles."""
    from oracle import regex_layer as rx
    torch, P = _env()
    g = gen.rng(99)
    alphabet = np.frombuffer(b"0123456789abcdef.:- CVElan", np.uint8)
    text = alphabet[g.integers(0, alphabet.size, 40000)].copy()
    plants = [b"10.1.2.3", b"CVE-2021-44228", b"de:ad:be:ef:00:01", b"0123456789abcdef0123456789abcdef", b"a.b.lan", b"1:2:3:4:5:6:7:8"]
    for k in range(900):
        pl = plants[k % len(plants)]
        pos = int(g.integers(0, text.size - 64))
        text[pos:pos + len(pl)] = np.frombuffer(pl, np.uint8)
        if k % 3:
            text[pos - 1 if pos else 0] = 32
            text[pos + len(pl)] = 32
    cuts = np.unique(np.concatenate([[0, text.size], g.integers(0, text.size, 200), [4096, 4097, 8191, 36000, 36000, 36001]]))
    cuts = np.sort(np.concatenate([cuts, cuts[5:25]]))                      # duplicates = empty records
    cuts = cuts[(cuts <= 15000) | (cuts >= 32000)]                         # one record of about 17 000 bytes
    want = rx.scan_records(text, cuts)
    assert len(want) > 300
    ctx = P.Context(0, workspace_bytes=64 << 20)
    for mm in (rx.MAX_MATCH, 20):
        R = P.Regex(ctx, _blob(mm))
        w = want if mm == rx.MAX_MATCH else rx.scan_records(text, cuts, max_match=mm)
        rc, n, got = _scan_gpu(torch, P, ctx, R, text, cuts, len(w) + 1)
        assert rc == 0 and n == len(w)
        assert np.array_equal(got, np.asarray(w, np.int32).reshape(-1, 4))
        R.close()
    # nothing to scan
    R = P.Regex(ctx, _blob())
    rc, n, got = _scan_gpu(torch, P, ctx, R, np.zeros(0, np.uint8), np.zeros(1, np.int64), 4)
    assert rc == 0 and n == 0
    rc, n, got = _scan_gpu(torch, P, ctx, R, np.zeros(0, np.uint8), np.zeros(5, np.int64), 4)
    assert rc == 0 and n == 0
    R.close(); ctx.close()


def test_regex_load_rejects_bad_tables():
    torch, P = _env()
    ctx = P.Context(0, workspace_bytes=1 << 20)
    blob = bytearray(_blob())
    for mutate in (lambda b: b.__setitem__(0, 0), lambda b: b.__setitem__(slice(-2, None), b"\xff\xff"), lambda b: b.append(0),
                   lambda b: b.__setitem__(32 + 5, 250)):
        bad = bytearray(blob)
        mutate(bad)
        with pytest.raises(P.AnonError):
            P.Regex(ctx, bytes(bad))
    ctx.close()


def _merge_gpu(torch, P, ctx, ner, rgx, cap, counts_on_device):
    dev = torch.device("cuda", 0)
    pad = 5 if counts_on_device else 0
    a = np.asarray(ner, np.int32).reshape(-1, 4)
    b = np.asarray(rgx, np.int32).reshape(-1, 4)
    d_a = torch.from_numpy(np.concatenate([a, np.full((pad, 4), 9999, np.int32)])).to(dev)
    d_b = torch.from_numpy(np.concatenate([b, np.full((pad, 4), 9999, np.int32)])).to(dev)
    na = torch.tensor([len(a)], dtype=torch.int32, device=dev) if counts_on_device else None
    nb = torch.tensor([len(b)], dtype=torch.int32, device=dev) if counts_on_device else None
    out = torch.full((max(cap, 1), 4), -7, dtype=torch.int32, device=dev)[:cap]
    num = torch.full((1,), -1, dtype=torch.int32, device=dev)
    P.anon_merge_spans(ctx, d_a, na, d_b, nb, out, num)
    rc = ctx.sync()
    n = int(num.item())
    return rc, n, out[:min(n, cap)].cpu().numpy()


def test_merge_matches_oracle():
    from oracle import decode, regex_layer as rx
    torch, P = _env()
    d, rec, _pool = _records(120, 47)
    win = gen.window_records(rec)
    ner = decode.decode_spans(win["planted_label"].astype(np.int32), win["meta"])
    rgx = rx.scan_records(rec["text"], rec["rec_off"])
    # NER spans that only partly agree with the regex spans: shift / shrink / drop some
    g = gen.rng(3)
    ner2 = []
    for (r, cs, ce, t) in ner:
        u = g.random()
        if u < 0.3:
            continue
        if u < 0.5 and ce - cs > 3:
            cs, ce = cs + 1, ce - 1
        ner2.append((r, cs, ce, t))
    # and an NER list that is unrelated to the regex spans: some spans clash, some touch, most stand alone
    ner_rand = []
    for r in range(len(rec["rec_off"]) - 1):
        n, pos = int(rec["rec_off"][r + 1] - rec["rec_off"][r]), 0
        while True:
            pos += int(g.integers(0, 120))
            wd = int(g.integers(1, 12))
            if pos + wd > n:
                break
            ner_rand.append((r, pos, pos + wd, int(g.integers(0, 4))))
            pos += wd
    assert len(ner2) > 1000 and len(rgx) > 1000 and len(ner_rand) > 1000
    ctx = P.Context(0, workspace_bytes=64 << 20)
    for lst in (ner2, ner_rand):
        want = rx.merge_spans(lst, rgx)
        if lst is ner_rand:
            assert len(rgx) + 100 < len(want) < len(rgx) + len(lst) - 100     # both outcomes occur
        for on_dev in (False, True):
            rc, n, got = _merge_gpu(torch, P, ctx, lst, rgx, len(lst) + len(rgx), on_dev)
            assert rc == 0 and n == len(want)
            assert np.array_equal(got, np.asarray(want, np.int32).reshape(-1, 4))
    # hand cases: touching spans are kept, overlapping dropped, one side empty, capacity
    ner3 = [(0, 0, 4, 1), (0, 10, 20, 2), (0, 30, 35, 0), (1, 5, 9, 3), (2, 0, 3, 1)]
    rgx3 = [(0, 15, 25, 4), (0, 35, 40, 5), (1, 0, 5, 0), (1, 8, 12, 0)]
    for a, b in ((ner3, rgx3), (ner3, []), ([], rgx3), ([], [])):
        w = rx.merge_spans(a, b)
        rc, n, got = _merge_gpu(torch, P, ctx, a, b, 16, True)
        assert rc == 0 and n == len(w) and np.array_equal(got, np.asarray(w, np.int32).reshape(-1, 4))
    rc, n, got = _merge_gpu(torch, P, ctx, ner3, rgx3, 3, False)
    assert rc == P.binding.ERR_CAPACITY and n == 7
    assert np.array_equal(got, np.asarray(rx.merge_spans(ner3, rgx3)[:3], np.int32))
    ctx.close()


def test_pipeline_with_regex_matches_oracle_composition():
    """The hybrid strategy end to end: NER spans from the FP32 tiny model merged with regex spans, pseudonymized
    and spliced -- spans, tokens, hit flags and the rewritten text equal the oracle's."""
    from oracle import crypto, decode, encoder, regex_layer as rx
    torch, P = _env()
    d, rec, _pool = _records(24, 5, median=250)
    win = gen.window_records(rec)
    w = gen.make_weights(d, gen.SEED_BASE + 1, planted=(2.0, 0.5, 4.0))
    key, names = bytes(range(1, 33)), gen.TYPE_NAMES_6
    logits = encoder.forward_packed(w, d, win["token_ids"], win["cu_seqlens"])
    assert encoder.top2_margin(logits).min() > 1e-3
    ner = decode.decode_spans(encoder.argmax_labels(logits), win["meta"])
    rgx = rx.scan_records(rec["text"], rec["rec_off"])
    spans = rx.merge_spans(ner, rgx)
    assert len(rgx) > 50 and len(spans) >= len(rgx)
    sb, so = decode.gather_spans(rec["text"], rec["rec_off"], spans)
    oc = crypto.Cache()
    want = oc.pseudonymize(sb, so, np.asarray([s[3] for s in spans], np.uint8), key, 10, names)
    oc.close()
    want_text, want_ro = decode.splice_records(rec["text"], rec["rec_off"], spans, want["out_tokens"], want["out_offsets"])

    ctx = P.Context(0, workspace_bytes=256 << 20)
    W = P.Weights(ctx, d, gen.pack_blob(w))
    cache = P.Cache(ctx, 4096, 1 << 20)
    R = P.Regex(ctx, _blob())
    P.anon_ctx_set_regex(ctx, R)
    T = win["token_ids"].size
    res = P.anon_pipeline_host(ctx, W, cache, win["token_ids"], win["cu_seqlens"], win["meta"], rec["text"], rec["rec_off"],
                               key, 10, names, span_capacity=T, out_capacity=T * 32, want_text=True)
    assert np.array_equal(res["spans"], np.asarray(spans, np.int32).reshape(-1, 4))
    assert np.array_equal(res["out_tokens"], want["out_tokens"]) and np.array_equal(res["hit"], want["hit"])
    assert np.array_equal(res["new_text"], want_text) and np.array_equal(res["new_record_offsets"], want_ro)
    # detached again: the plain NER path
    P.anon_ctx_set_regex(ctx, None)
    cache.clear()
    res = P.anon_pipeline_host(ctx, W, cache, win["token_ids"], win["cu_seqlens"], win["meta"], rec["text"], rec["rec_off"],
                               key, 10, names, span_capacity=T, out_capacity=T * 32)
    assert np.array_equal(res["spans"], np.asarray(ner, np.int32).reshape(-1, 4))
    R.close(); cache.close(); W.close(); ctx.close()


def test_two_automata_of_different_size_side_by_side():
    """A small automaton loaded after a large one must not shrink what the large one may launch with (both share one kernel)."""
    from oracle import regex_layer as rx
    from paper_2606_15650_b200 import regex_dfa
    torch, P = _env()
    d, rec, _pool = _records(30, 71)
    text, off = rec["text"], rec["rec_off"]
    one = [("CVE_ID", rx.PATTERNS[3][1])]
    ctx = P.Context(0, workspace_bytes=64 << 20)
    big = P.Regex(ctx, _blob())
    small = P.Regex(ctx, regex_dfa.compile_patterns([(3, one[0][1])], rx.MAX_MATCH))
    for R, pats in ((big, rx.PATTERNS), (small, one), (big, rx.PATTERNS)):
        want = rx.scan_records(text, off, pats)
        if pats is one:
            want = [(r, a, b, 3) for r, a, b, _k in want]            # the automaton reports the type id given at compile time
        rc, n, got = _scan_gpu(torch, P, ctx, R, text, off, len(want) + 4)
        assert rc == 0 and n == len(want) and n > 5
        assert np.array_equal(got, np.asarray(want, np.int32).reshape(-1, 4))
    small.close(); big.close(); ctx.close()


def test_random_pattern_sets_match_oracle():
    """Fuzz on the device: 40 random pattern sets of the restricted grammar (different automaton sizes, class counts, type
    maps and max_match), random text over a small alphabet cut into ragged records; spans bit-exact against the oracle."""
    import re
    from oracle import regex_layer as rx
    from paper_2606_15650_b200 import regex_dfa
    from test_regex_dfa import _random_pattern
    torch, P = _env()
    rng = np.random.default_rng(77)
    alphabet = np.frombuffer(b"abc01.- x", np.uint8)
    ctx = P.Context(0, workspace_bytes=64 << 20)
    done = 0
    while done < 40:
        pats = [_random_pattern(rng) for _ in range(int(rng.integers(1, 5)))]
        if any(re.fullmatch(p, "") for p in pats):
            continue
        mm = int(rng.integers(3, 40))
        types = [int(rng.integers(0, 9)) for _ in pats]
        R = P.Regex(ctx, regex_dfa.compile_patterns(list(zip(types, pats)), mm))
        text = alphabet[rng.integers(0, alphabet.size, 9000)].copy()
        cuts = np.unique(np.concatenate([[0, text.size], rng.integers(0, text.size, 25)]))
        want = [(r, a, b, types[k]) for r, a, b, k in rx.scan_records(text, cuts, [("P", p) for p in pats], mm)]
        rc, n, got = _scan_gpu(torch, P, ctx, R, text, cuts, len(want) + 2)
        assert rc == 0 and n == len(want), (pats, mm)
        assert np.array_equal(got, np.asarray(want, np.int32).reshape(-1, 4)), (pats, mm)
        R.close()
        done += 1
    ctx.close()
