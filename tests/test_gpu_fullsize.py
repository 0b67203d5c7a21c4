"""GPU parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times (one ~1 M-token chunk for
configs[1]; 50 M spans in one call for configs[4]).  The oracle cannot run these sizes whole, so:
  * encoder: oracle logits / labels on sampled sequences (computed one by one), BF16 tolerances of BASELINE.json;
  * decode / gather / pseudonymize: the oracle applied to the GPU's own labels and spans (those stages are integer
    work: bit-exact at full size);
  * configs[4]: the hit / miss sets and uids follow from the generator's draws alone (first occurrence of each string),
    the pseudonyms of sampled spans come from the oracle's HMAC one by one."""
import numpy as np
import pytest

from harness import gen

pytestmark = pytest.mark.gpu

KEY = bytes((7 * i + 3) & 255 for i in range(32))


def test_configs1_full_size_in_bench_configuration():
    import torch
    import paper_2606_15650_b200 as P
    from oracle import crypto, decode, encoder
    if not torch.cuda.is_available():
        pytest.fail("GPU test selected but no CUDA device")
    dev = "cuda:0"
    d = gen.DESCS["base"]
    rec, win = gen.workload_base(n_records=4096, seed=gen.SEED_BASE + 2)          # exactly bench.py's default workload
    w = gen.make_weights(d, gen.SEED_BASE + 2, planted=(2.0, 0.5, 4.0))
    ids, cu, meta = win["token_ids"], win["cu_seqlens"], np.ascontiguousarray(win["meta"])
    T, B = ids.size, cu.size - 1
    assert T > 900_000
    ctx = P.Context(0, workspace_bytes=P.anon_workspace_bytes(d, T, B) + (256 << 20))
    W = P.Weights(ctx, d, gen.pack_blob(w))
    logits = torch.zeros((T, d["num_labels"]), dtype=torch.float32, device=dev)
    labels = torch.zeros(T, dtype=torch.int32, device=dev)
    P.anon_ner_forward(ctx, W, torch.from_numpy(ids).to(dev), torch.from_numpy(cu).to(dev), logits, labels)
    assert ctx.sync() == 0
    got_logits, got_labels = logits.cpu().numpy(), labels.cpu().numpy()
    # the GPU label is the argmax (ties -> lowest) of the GPU's own FP32 logits, everywhere
    assert np.array_equal(got_labels, encoder.argmax_labels(got_logits))
    # sampled sequences: shortest, longest, first, last, and four seeded picks (tiles in the middle of the launch)
    lens = np.diff(cu)
    picks = {int(np.argmin(lens)), int(np.argmax(lens)), 0, B - 1}
    picks |= set(np.random.default_rng(5).integers(0, B, 4).tolist())
    subset = sorted(picks)
    want = encoder.forward_packed(w, d, ids, cu, seq_subset=subset)
    rows = ~np.isnan(want[:, 0])
    assert rows.sum() >= 512
    err = np.abs(got_logits[rows] - want[rows])
    assert err.max() <= 3e-2, err.max()
    mism = got_labels[rows] != encoder.argmax_labels(want[rows])
    assert (encoder.top2_margin(want[rows])[mism] < 3e-2).all()
    assert 1.0 - mism.mean() >= 0.999
    # decode + gather + pseudonymize at full size against the oracle fed with the GPU's labels
    cap = T // 2
    spans = torch.zeros((cap, 4), dtype=torch.int32, device=dev)
    nsp = torch.zeros(1, dtype=torch.int32, device=dev)
    P.anon_decode_spans(ctx, labels, torch.from_numpy(meta).to(dev), d["num_labels"], spans, nsp)
    assert ctx.sync() == 0
    S = int(nsp.item())
    want_spans = decode.decode_spans(got_labels, meta)
    assert S == len(want_spans) and S > 20000
    assert np.array_equal(spans.cpu().numpy()[:S], np.asarray(want_spans, np.int32).reshape(-1, 4))
    text, rec_off = rec["text"], rec["rec_off"]
    span_bytes = torch.zeros(text.size + 16, dtype=torch.uint8, device=dev)
    span_off = torch.zeros(S + 1, dtype=torch.int64, device=dev)
    span_type = torch.zeros(S, dtype=torch.uint8, device=dev)
    P.anon_gather_spans(ctx, torch.from_numpy(text).to(dev), torch.from_numpy(rec_off).to(dev), spans, S, span_bytes, span_off,
                        span_type)
    sb, so = decode.gather_spans(text, rec_off, want_spans)
    assert ctx.sync() == 0
    assert np.array_equal(span_off.cpu().numpy(), so) and np.array_equal(span_bytes.cpu().numpy()[:so[-1]], sb)
    cache = P.Cache(ctx, 1 << 20, 64 << 20)
    out = torch.zeros(S * 32, dtype=torch.uint8, device=dev)
    out_off = torch.zeros(S + 1, dtype=torch.int64, device=dev)
    hit = torch.zeros(S, dtype=torch.uint8, device=dev)
    P.anon_pseudonymize(ctx, cache, span_bytes, span_off, span_type, KEY, 10, gen.TYPE_NAMES_6, out, out_off, hit)
    assert ctx.sync() == 0
    oc = crypto.Cache(1 << 20)
    wantp = oc.pseudonymize(sb, so, np.asarray([s[3] for s in want_spans], np.uint8), KEY, 10, gen.TYPE_NAMES_6)
    oc.close()
    oo = out_off.cpu().numpy()
    assert np.array_equal(oo, wantp["out_offsets"])
    assert np.array_equal(out.cpu().numpy()[:oo[-1]], wantp["out_tokens"])
    assert np.array_equal(hit.cpu().numpy(), wantp["hit"])
    cache.close(); W.close(); ctx.close()


def test_configs2_stream_subsample():
    """BASELINE.json configs[2] at its real shape (the workload stands in for the paper's D2,
    PAPER.md L111: 70,951 records / 550 MB): the first 64 records of bench.py's stream (same seeds, same 300 k-string
    Zipf pool, so these ARE the stream's first 64 records) with ALL their windows, BERT-base shape BF16, deep planted
    detector, run through anon_pipeline_host_text in >= 3 token-budgeted batches with ONE persistent cache.
      * oracle encoder (fp64) on every window: logits max-abs <= 3e-2; labels >= 99.9 % equal, every mismatch at oracle
        top-2 margin < 3e-2;
      * oracle decode of the GPU's labels == GPU spans, bit-exact, spans crossing a window boundary included;
      * oracle dedup / HMAC / write-back / splice of the GPU span list == GPU tokens, hit flags and rewritten text;
      * planted-truth recall and spans / planted are printed (and must be sane)."""
    import torch
    import paper_2606_15650_b200 as P
    from paper_2606_15650_b200 import stream
    from oracle import crypto, decode, encoder
    if not torch.cuda.is_available():
        pytest.fail("GPU test selected but no CUDA device")
    dev = "cuda:0"
    d = gen.DESCS["base"]
    rec = gen.workload_stream(n_records=64, seed=gen.SEED_BASE + 3, n_pool=300000)
    win = gen.window_records(rec)
    w = gen.make_weights(d, gen.SEED_BASE + 2, planted=gen.PLANTED_DEEP)
    ids, cu, meta = win["token_ids"], win["cu_seqlens"], np.ascontiguousarray(win["meta"])
    T, B = ids.size, cu.size - 1
    assert T > 100_000 and B > 250 and np.diff(cu).max() == 512
    plan = stream.plan_batches(win["win_rec"], cu, T // 4)
    assert len(plan) >= 3
    maxT = max(int(cu[b] - cu[a]) for a, b in plan)
    ctx = P.Context(0, workspace_bytes=P.anon_workspace_bytes(d, T, B) + 200 * T + 4 * rec["text"].size + (256 << 20))
    W = P.Weights(ctx, d, gen.pack_blob(w))
    logits = torch.zeros((T, d["num_labels"]), dtype=torch.float32, device=dev)
    labels = torch.zeros(T, dtype=torch.int32, device=dev)
    P.anon_ner_forward(ctx, W, torch.from_numpy(ids).to(dev), torch.from_numpy(cu).to(dev), logits, labels)
    assert ctx.sync() == 0
    got_logits, got_labels = logits.cpu().numpy(), labels.cpu().numpy()
    cache = P.Cache(ctx, 1 << 18, 16 << 20)
    got_spans, got_tok, got_hit, got_len, got_text, got_ro = [], [], [], [], [], []
    for a, b in plan:
        bt = stream.slice_batch(rec, win, a, b)
        res = P.anon_pipeline_host(ctx, W, cache, bt["token_ids"], bt["cu_seqlens"], bt["meta"], bt["text"], bt["rec_off"], KEY, 10,
                                   gen.TYPE_NAMES_6, span_capacity=maxT // 4, out_capacity=maxT * 8, want_text=True)
        sp = res["spans"].copy()
        sp[:, 0] += bt["r0"]
        got_spans.append(sp)
        got_tok.append(res["out_tokens"].copy())
        got_hit.append(res["hit"].copy())
        got_len.append(np.diff(res["out_offsets"]))
        got_text.append(res["new_text"].copy())
        got_ro.append(np.diff(res["new_record_offsets"]))
    st = cache.stats()
    cache.close(); W.close(); ctx.close()
    got_spans = np.concatenate(got_spans)
    # ---- encoder against the fp64 oracle, every window ----
    want = encoder.forward_packed(w, d, ids, cu)
    err = np.abs(got_logits - want)
    assert err.max() <= 3e-2, err.max()
    want_labels = encoder.argmax_labels(want)
    mism = got_labels != want_labels
    assert (encoder.top2_margin(want)[mism] < 3e-2).all()
    assert 1.0 - mism.mean() >= 0.999
    assert np.array_equal(got_labels, encoder.argmax_labels(got_logits))
    # ---- decode: the oracle walk over the GPU's labels (batch by batch == the undivided stream) ----
    spans = decode.decode_spans(got_labels, meta)
    assert np.array_equal(got_spans, np.asarray(spans, np.int32).reshape(-1, 4))
    # at least one span is stitched across a window boundary: its kept tokens lie in two windows
    win_of_tok = np.repeat(np.arange(B), np.diff(cu))
    kept = meta[:, 3] == 1
    first_tok = {}
    for j in np.flatnonzero(kept & (got_labels > 0)):
        first_tok.setdefault((int(meta[j, 0]), int(meta[j, 1])), j)
    crossing = 0
    for r, cs, ce, _t in spans:
        j = first_tok[(r, cs)]
        k = j
        while not (kept[k] and meta[k, 0] == r and meta[k, 2] == ce):
            k += 1
        crossing += int(win_of_tok[k] != win_of_tok[j])
    assert crossing >= 1
    # ---- dedup / HMAC / write-back / splice on the GPU span list ----
    sb, so = decode.gather_spans(rec["text"], rec["rec_off"], spans)
    oc = crypto.Cache(1 << 18)
    wantp = oc.pseudonymize(sb, so, np.asarray([s[3] for s in spans], np.uint8), KEY, 10, gen.TYPE_NAMES_6)
    oc.close()
    assert np.array_equal(np.concatenate(got_tok), wantp["out_tokens"])
    assert np.array_equal(np.concatenate(got_hit), wantp["hit"])
    assert np.array_equal(np.concatenate(got_len), np.diff(wantp["out_offsets"]))
    assert st["n_lookups"] == len(spans) and st["n_hits"] == int(wantp["hit"].sum()) and wantp["hit"].sum() > 0
    want_text, want_ro = decode.splice_records(rec["text"], rec["rec_off"], spans, wantp["out_tokens"], wantp["out_offsets"])
    assert np.array_equal(np.concatenate(got_text), want_text)
    assert np.array_equal(np.concatenate(got_ro), np.diff(want_ro))
    # ---- planted truth (a report; the oracle's labels stay the parity reference) ----
    planted = set(decode.decode_spans(win["planted_label"].astype(np.int32), meta))
    found = set(spans)
    recall = len(planted & found) / len(planted)
    print(f"configs[2] subsample: T={T} windows={B} batches={len(plan)} spans={len(spans)} planted={len(planted)} "
          f"spans/planted={len(spans) / len(planted):.4f} recall={recall:.4f} crossing={crossing} max|dlogit|={err.max():.2e} "
          f"label mismatches={int(mism.sum())} hit rate={st['n_hits'] / st['n_lookups']:.3f}")
    assert len(planted) == rec["n_entities"] and recall >= 0.99 and len(spans) <= 1.01 * len(planted)


def test_configs4_full_size_50m_spans():
    import torch
    import paper_2606_15650_b200 as P
    from oracle import crypto
    if not torch.cuda.is_available():
        pytest.fail("GPU test selected but no CUDA device")
    dev = "cuda:0"
    n_unique, S = 2_000_000, 50_000_000
    data, off, types, key, draws = gen.spans_zipf(n_unique, S, 7, 128, 6, gen.SEED_BASE + 5)      # bench.py's workload
    ctx = P.Context(0, workspace_bytes=S * 9 + (S // 2048 + 2) * 24 + (64 << 20))
    cache = P.Cache(ctx, n_unique, int(n_unique * 70) + (1 << 20))
    d_bytes, d_off, d_type = (torch.from_numpy(a).to(dev) for a in (data, off, types))
    out = torch.zeros(S * (3 + 13 + 10), dtype=torch.uint8, device=dev)
    out_off = torch.zeros(S + 1, dtype=torch.int64, device=dev)
    hit = torch.zeros(S, dtype=torch.uint8, device=dev)
    uid = torch.zeros(S, dtype=torch.int64, device=dev)
    kb = key.tobytes()
    P.anon_pseudonymize(ctx, cache, d_bytes, d_off, d_type, kb, 10, gen.TYPE_NAMES_6, out, out_off, hit, uid)
    assert ctx.sync() == 0
    # hit / miss sets and uids from the draws alone: a span misses iff it is the first occurrence of its pool string,
    # and uid = rank of that first occurrence among all first occurrences (the pool strings are distinct by construction)
    _vals, first = np.unique(draws, return_index=True)
    want_hit = np.ones(S, np.uint8)
    want_hit[first] = 0
    got_hit = hit.cpu().numpy()
    assert np.array_equal(got_hit, want_hit)
    order = np.sort(first)                                   # first occurrences in stream order -> uid 0, 1, 2, ...
    uid_of_pool = np.empty(n_unique, np.int64)
    uid_of_pool[draws[order]] = np.arange(order.size)
    assert np.array_equal(uid.cpu().numpy(), uid_of_pool[draws])
    st = cache.stats()
    assert st["n_unique"] == first.size and st["n_lookups"] == S and st["n_hits"] == S - first.size
    # offsets: exclusive prefix sum of 3 + len(type name) + slug_len
    name_len = np.asarray([len(n) for n in gen.TYPE_NAMES_6], np.int64)
    want_off = np.zeros(S + 1, np.int64)
    np.cumsum(3 + name_len[types] + 10, out=want_off[1:])
    got_off = out_off.cpu().numpy()
    assert np.array_equal(got_off, want_off)
    # sampled pseudonyms from the oracle, one by one: the first and last spans, the head of the Zipf law, seeded picks
    picks = np.unique(np.concatenate([[0, 1, S - 1], order[:50], np.random.default_rng(9).integers(0, S, 4000)]))
    got_tok = out.cpu().numpy()
    sub_off = np.zeros(picks.size + 1, np.int64)
    np.cumsum(off[picks + 1] - off[picks], out=sub_off[1:])
    sub = np.concatenate([data[off[i]:off[i + 1]] for i in picks])
    dig = crypto.hmac_batch(kb, sub, sub_off)
    for k, i in enumerate(picks):
        want_tok = ("[" + gen.TYPE_NAMES_6[types[i]] + "_" + bytes(dig[k]).hex()[:10] + "]").encode()
        assert bytes(got_tok[got_off[i]:got_off[i + 1]]) == want_tok, int(i)
    cache.close(); ctx.close()


def test_configs3_full_size_in_bench_configuration():
    """BASELINE.json configs[3] at the size `bench.py --workload large` times: 16,384 packed sequences U[32, 512]
    (~4.45 M tokens) through the 24 x 1024 encoder with the 250,002-row embedding table, in one `anon_ner_forward`
    call.  Oracle logits / labels on sampled sequences (shortest, longest, last, one seeded pick); labels == argmax of
    the GPU's own logits on every token; decode bit-exact against the oracle fed with the GPU's labels."""
    import torch
    import paper_2606_15650_b200 as P
    from oracle import decode, encoder
    if not torch.cuda.is_available():
        pytest.fail("GPU test selected but no CUDA device")
    dev = "cuda:0"
    d = gen.DESCS["large"]
    rec, win = gen.workload_large(n_seqs=16384, seed=gen.SEED_BASE + 4)             # exactly bench.py's "large" workload
    w = gen.make_weights(d, gen.SEED_BASE + 4, planted=gen.PLANTED_DEEP)       # the 3-tuple plant fades to 0 spans at L = 24
    ids, cu, meta = win["token_ids"], win["cu_seqlens"], np.ascontiguousarray(win["meta"])
    T, B = ids.size, cu.size - 1
    assert B == 16384 and T > 4_000_000
    ctx = P.Context(0, workspace_bytes=P.anon_workspace_bytes(d, T, B) + (256 << 20))
    W = P.Weights(ctx, d, gen.pack_blob(w))
    logits = torch.zeros((T, d["num_labels"]), dtype=torch.float32, device=dev)
    labels = torch.zeros(T, dtype=torch.int32, device=dev)
    P.anon_ner_forward(ctx, W, torch.from_numpy(ids).to(dev), torch.from_numpy(cu).to(dev), logits, labels)
    assert ctx.sync() == 0
    got_logits, got_labels = logits.cpu().numpy(), labels.cpu().numpy()
    assert np.array_equal(got_labels, encoder.argmax_labels(got_logits))
    cap = T // 2
    spans = torch.zeros((cap, 4), dtype=torch.int32, device=dev)
    nsp = torch.zeros(1, dtype=torch.int32, device=dev)
    P.anon_decode_spans(ctx, labels, torch.from_numpy(meta).to(dev), d["num_labels"], spans, nsp)
    assert ctx.sync() == 0
    S = int(nsp.item())
    got_spans = spans.cpu().numpy()[:S]
    assert S > 100_000                          # ~1 entity per 25 tokens: A9-A13 are exercised at this shape
    # gather + pseudonymize at full size, checked below against the oracle fed with the GPU's spans
    text, rec_off = rec["text"], rec["rec_off"]
    span_bytes = torch.zeros(text.size + 16, dtype=torch.uint8, device=dev)
    span_off = torch.zeros(S + 1, dtype=torch.int64, device=dev)
    span_type = torch.zeros(S, dtype=torch.uint8, device=dev)
    P.anon_gather_spans(ctx, torch.from_numpy(text).to(dev), torch.from_numpy(rec_off).to(dev), spans, S, span_bytes, span_off,
                        span_type)
    cache = P.Cache(ctx, 1 << 20, 64 << 20)
    out = torch.zeros(S * 32, dtype=torch.uint8, device=dev)
    out_off = torch.zeros(S + 1, dtype=torch.int64, device=dev)
    hit = torch.zeros(S, dtype=torch.uint8, device=dev)
    P.anon_pseudonymize(ctx, cache, span_bytes, span_off, span_type, KEY, 10, gen.TYPE_NAMES_6, out, out_off, hit)
    assert ctx.sync() == 0
    got_sb, got_so, got_oo, got_out, got_hit = (t.cpu().numpy() for t in (span_bytes, span_off, out_off, out, hit))
    cache.close(); W.close(); ctx.close()
    want_spans = decode.decode_spans(got_labels, meta)
    assert S == len(want_spans)
    assert np.array_equal(got_spans, np.asarray(want_spans, np.int32).reshape(-1, 4))
    sb, so = decode.gather_spans(text, rec_off, want_spans)
    assert np.array_equal(got_so, so) and np.array_equal(got_sb[:so[-1]], sb)
    from oracle import crypto
    oc = crypto.Cache(1 << 20)
    wantp = oc.pseudonymize(sb, so, np.asarray([s[3] for s in want_spans], np.uint8), KEY, 10, gen.TYPE_NAMES_6)
    oc.close()
    assert np.array_equal(got_oo, wantp["out_offsets"]) and np.array_equal(got_out[:got_oo[-1]], wantp["out_tokens"])
    assert np.array_equal(got_hit, wantp["hit"])
    planted = set(decode.decode_spans(win["planted_label"].astype(np.int32), meta))
    print(f"configs[3]: T={T} spans={S} planted={len(planted)} recall={len(planted & set(want_spans)) / len(planted):.4f}")
    lens = np.diff(cu)
    picks = {int(np.argmin(lens)), int(np.argmax(lens)), B - 1} | set(np.random.default_rng(7).integers(0, B, 1).tolist())
    want = encoder.forward_packed(w, d, ids, cu, seq_subset=sorted(picks))
    rows = ~np.isnan(want[:, 0])
    assert rows.sum() >= 512
    err = np.abs(got_logits[rows] - want[rows])
    assert err.max() <= 3e-2, err.max()
    mism = got_labels[rows] != encoder.argmax_labels(want[rows])
    assert (encoder.top2_margin(want[rows])[mism] < 3e-2).all()
    assert 1.0 - mism.mean() >= 0.999


def test_modern_shape_full_size_in_bench_configuration():
    """NEXT-3 at the size `bench.py --workload modern` times: 4096 records, ~1 M tokens in one chunk through the 22-layer
    ModernBERT-base-shaped encoder; oracle logits / labels on sampled sequences (shortest, longest, first, last, seeded picks)."""
    import torch
    import paper_2606_15650_b200 as P
    from oracle import encoder, encoder_modern
    if not torch.cuda.is_available():
        pytest.fail("GPU test selected but no CUDA device")
    dev = "cuda:0"
    d = gen.DESCS["base_modern"]
    rec, win = gen.workload_base(n_records=4096, seed=gen.SEED_BASE + 2, desc=d)    # bench.py's "modern" workload
    w = gen.make_weights_modern(d, gen.SEED_BASE + 7, planted=(2.0, 0.5, 4.0))
    ids, cu = win["token_ids"], win["cu_seqlens"]
    T, B = ids.size, cu.size - 1
    assert T > 900_000
    ctx = P.Context(0, workspace_bytes=P.anon_workspace_bytes(d, T, B) + (256 << 20))
    W = P.Weights(ctx, d, gen.pack_blob_modern(w))
    logits = torch.zeros((T, d["num_labels"]), dtype=torch.float32, device=dev)
    labels = torch.zeros(T, dtype=torch.int32, device=dev)
    P.anon_ner_forward(ctx, W, torch.from_numpy(ids).to(dev), torch.from_numpy(cu).to(dev), logits, labels)
    assert ctx.sync() == 0
    got_logits, got_labels = logits.cpu().numpy(), labels.cpu().numpy()
    W.close(); ctx.close()
    assert np.array_equal(got_labels, encoder.argmax_labels(got_logits))
    lens = np.diff(cu)
    picks = {int(np.argmin(lens)), int(np.argmax(lens)), 0, B - 1} | set(np.random.default_rng(6).integers(0, B, 3).tolist())
    want = encoder_modern.forward_packed(w, d, ids, cu, seq_subset=sorted(picks))
    rows = ~np.isnan(want[:, 0])
    assert rows.sum() >= 512
    err = np.abs(got_logits[rows] - want[rows])
    assert err.max() <= 3e-2, err.max()
    mism = got_labels[rows] != encoder.argmax_labels(want[rows])
    assert (encoder.top2_margin(want[rows])[mism] < 3e-2).all()
    assert 1.0 - mism.mean() >= 0.999


def test_regex_scan_full_size():
    """NEXT-4 at the size kernel_bench times (~400 MB of configs[2]-shaped text, one call): the oracle's brute-force scan on
    sampled records (first, last, longest, seeded picks) equals the GPU's spans for those records; over ALL spans: ordered,
    inside their record, non-overlapping, word-bounded, and `re.fullmatch` of the reported pattern on a seeded sample."""
    import re
    import torch
    import paper_2606_15650_b200 as P
    from oracle import regex_layer as rx
    from paper_2606_15650_b200 import regex_dfa
    if not torch.cuda.is_available():
        pytest.fail("GPU test selected but no CUDA device")
    dev = "cuda:0"
    rec = gen.workload_stream(n_records=2000, n_pool=50000)
    reps = int(400e6 / rec["text"].size)
    text = np.tile(rec["text"], reps)
    sizes = np.tile(np.diff(rec["rec_off"]), reps)
    roff = np.zeros(sizes.size + 1, np.int64)
    roff[1:] = np.cumsum(sizes)
    R = sizes.size
    ctx = P.Context(0, workspace_bytes=int(text.size * 2.2) + (64 << 20))
    rgx = P.Regex(ctx, regex_dfa.compile_patterns([(k, p) for k, (_n, p) in enumerate(rx.PATTERNS)], rx.MAX_MATCH))
    cap = text.size // 40
    spans = torch.zeros((cap, 4), dtype=torch.int32, device=dev)
    num = torch.zeros(1, dtype=torch.int32, device=dev)
    P.anon_regex_scan(ctx, rgx, torch.from_numpy(text).to(dev), torch.from_numpy(roff).to(dev), spans, num)
    assert ctx.sync() == 0
    n = int(num.item())
    got = spans[:n].cpu().numpy()
    rgx.close(); ctx.close()
    assert 1_000_000 < n <= cap
    r, cs, ce, k = got[:, 0].astype(np.int64), got[:, 1].astype(np.int64), got[:, 2].astype(np.int64), got[:, 3]
    assert (np.diff(r) >= 0).all() and (cs < ce).all() and (ce - cs <= rx.MAX_MATCH).all() and (ce <= sizes[r]).all()
    same = np.diff(r) == 0
    assert (cs[1:][same] >= ce[:-1][same]).all()                                   # non-overlapping, ordered inside a record
    word = np.zeros(256, bool); word[list(rx._WORD)] = True
    a, b = roff[r] + cs, roff[r] + ce
    inner = cs > 0
    assert not word[text[a[inner] - 1]].any()                                      # left word boundary
    inner = ce < sizes[r]
    assert not word[text[b[inner]]].any()                                          # right word boundary
    for i in np.random.default_rng(8).integers(0, n, 3000):
        assert re.fullmatch(rx.PATTERNS[k[i]][1].encode(), text[a[i]:b[i]].tobytes())
    picks = {0, R - 1, int(np.argmax(sizes))} | set(np.random.default_rng(9).integers(0, R, 40).tolist())
    for q in sorted(picks):
        want = rx.scan_record(text[roff[q]:roff[q + 1]].tobytes())
        lo, hi = np.searchsorted(r, q), np.searchsorted(r, q, side="right")
        assert [tuple(x) for x in got[lo:hi, 1:].tolist()] == want, q
