"""Streaming in token-budgeted batches (BASELINE.json configs[2] shape).

CPU part: the batch plan covers every window once, cuts only between records, respects the budget, and a sliced
batch is a self-contained input (oracle decode of the slices == oracle decode of the whole stream).
GPU part: the whole hot path run batch by batch through anon_pipeline_host with a persistent cache equals the
oracle run over the undivided stream -- spans, pseudonyms and hit flags bit-exact (referential integrity across
batches, PAPER.md L38 / L50)."""
import numpy as np
import pytest

from harness import gen
from paper_2606_15650_b200 import stream


def _small_stream(n_records=40, seed=7):
    d = dict(gen.DESCS["tiny"])
    pool, poff, ptype = gen.entity_pool(48, seed)
    ptype = ptype % 4
    g = gen.rng(seed + 1)
    n_tok = np.minimum(g.lognormal(np.log(300), 1.0, n_records), 2500).astype(np.int64) + 8
    rec = gen.make_records(n_records, n_tok, d, pool, poff, ptype, seed + 2, zipf_s=1.1)
    win = gen.window_records(rec)
    return d, rec, win


def test_plan_covers_stream_and_cuts_between_records():
    d, rec, win = _small_stream()
    cu = win["cu_seqlens"]
    for budget in (600, 3000, 10 ** 9):
        plan = stream.plan_batches(win["win_rec"], cu, budget)
        assert plan[0][0] == 0 and plan[-1][1] == len(cu) - 1
        for (a0, a1), (b0, b1) in zip(plan[:-1], plan[1:]):
            assert a1 == b0 and a0 < a1
            assert win["win_rec"][a1 - 1] != win["win_rec"][b0]          # the cut is a record boundary
        for a, b in plan:
            nrec = len(set(win["win_rec"][a:b].tolist()))
            assert cu[b] - cu[a] <= budget or nrec == 1                    # only a single huge record may exceed
    assert len(stream.plan_batches(win["win_rec"], cu, 10 ** 9)) == 1
    assert stream.plan_batches(np.zeros(0, np.int32), np.zeros(1, np.int32), 100) == []


def test_sliced_batches_decode_like_the_whole_stream():
    from oracle import decode
    d, rec, win = _small_stream(seed=11)
    labels = win["planted_label"].astype(np.int32)                         # labels supplied directly
    whole = decode.decode_spans(labels, win["meta"])
    sb_w, so_w = decode.gather_spans(rec["text"], rec["rec_off"], whole)
    got_spans, got_bytes = [], []
    for a, b in stream.plan_batches(win["win_rec"], win["cu_seqlens"], 2500):
        bt = stream.slice_batch(rec, win, a, b)
        assert bt["cu_seqlens"][0] == 0 and bt["cu_seqlens"][-1] == bt["token_ids"].size
        assert bt["rec_off"][0] == 0 and bt["rec_off"][-1] == bt["text"].size
        assert bt["meta"][:, 0].min() >= 0 and bt["meta"][:, 0].max() < bt["rec_off"].size - 1
        sp = decode.decode_spans(labels[bt["t0"]:bt["t1"]], bt["meta"])
        sb, so = decode.gather_spans(bt["text"], bt["rec_off"], sp)
        got_spans += [(r + bt["r0"], cs, ce, t) for r, cs, ce, t in sp]
        got_bytes.append(sb)
    assert got_spans == [tuple(s) for s in whole]
    assert np.array_equal(np.concatenate(got_bytes), sb_w)


@pytest.mark.gpu
def test_stream_batches_match_oracle_on_gpu():
    import torch
    import paper_2606_15650_b200 as P
    from oracle import crypto, decode, encoder
    if not torch.cuda.is_available():
        pytest.fail("GPU test selected but no CUDA device")
    d, rec, win = _small_stream(n_records=24, seed=5)
    w = gen.make_weights(d, gen.SEED_BASE + 1, planted=(2.0, 0.5, 4.0))
    key, names = bytes(range(1, 33)), gen.TYPE_NAMES_4
    # oracle over the undivided stream
    logits = encoder.forward_packed(w, d, win["token_ids"], win["cu_seqlens"])
    labels = encoder.argmax_labels(logits)
    assert encoder.top2_margin(logits).min() > 1e-3                       # FP32 path: labels are then decided identically
    spans = decode.decode_spans(labels, win["meta"])
    sb, so = decode.gather_spans(rec["text"], rec["rec_off"], spans)
    oc = crypto.Cache()
    want = oc.pseudonymize(sb, so, np.asarray([s[3] for s in spans], np.uint8), key, 10, names)
    oc.close()
    assert len(spans) > 50 and want["hit"].sum() > 10                      # the cache is exercised across batches

    plan = stream.plan_batches(win["win_rec"], win["cu_seqlens"], 3000)
    assert len(plan) >= 3
    ctx = P.Context(0, workspace_bytes=256 << 20)
    W = P.Weights(ctx, d, gen.pack_blob(w))
    cache = P.Cache(ctx, 4096, 1 << 20)
    got_spans, got_tok, got_hit, got_len, got_text, got_ro = [], [], [], [], [], []
    for a, b in plan:
        bt = stream.slice_batch(rec, win, a, b)
        T = bt["token_ids"].size
        res = P.anon_pipeline_host(ctx, W, cache, bt["token_ids"], bt["cu_seqlens"], bt["meta"], bt["text"], bt["rec_off"],
                                   key, 10, names, span_capacity=T, out_capacity=T * 32, want_text=True)
        got_text.append(res["new_text"].copy())
        got_ro.append(res["new_record_offsets"].copy())
        sp = res["spans"].copy()
        sp[:, 0] += bt["r0"]
        got_spans.append(sp)
        got_tok.append(res["out_tokens"].copy())
        got_hit.append(res["hit"].copy())
        got_len.append(np.diff(res["out_offsets"]))
    st = cache.stats()
    cache.close(); W.close(); ctx.close()
    assert np.array_equal(np.concatenate(got_spans), np.asarray(spans, np.int32).reshape(-1, 4))
    assert np.array_equal(np.concatenate(got_tok), want["out_tokens"])
    assert np.array_equal(np.concatenate(got_hit), want["hit"])
    assert np.array_equal(np.concatenate(got_len), np.diff(want["out_offsets"]))
    assert st["n_lookups"] == len(spans) and st["n_hits"] == int(want["hit"].sum())
    # text in -> text out: the batches' rewritten records, concatenated, are the oracle's splice of the whole stream
    want_text, want_ro = decode.splice_records(rec["text"], rec["rec_off"], spans, want["out_tokens"], want["out_offsets"])
    assert np.array_equal(np.concatenate(got_text), want_text)
    sizes = np.concatenate([np.diff(r) for r in got_ro])
    assert np.array_equal(sizes, np.diff(want_ro))
