"""Host-side generator checks (CPU only): layout facts the hot path relies on."""
import numpy as np
import torch

from harness import gen
from oracle import decode


def test_bf16_round_matches_torch():
    a = (np.random.default_rng(0).standard_normal(10000) * 0.02).astype(np.float32)
    a[:4] = [0.0, 1.0, -1.0, 1.00390625]   # last one is a tie
    want = torch.tensor(a).to(torch.bfloat16).to(torch.float32).numpy()
    assert np.array_equal(gen.bf16_round(a), want)


def test_blob_order_and_size():
    d = gen.DESCS["tiny"]
    w = gen.make_weights(d, 1)
    blob = gen.pack_blob(w)
    H, F, V, NL, P, L = d["hidden"], d["ffn"], d["vocab"], d["num_labels"], d["max_pos"], d["layers"]
    per_layer = 3 * H * H + 3 * H + H * H + H + 2 * H + F * H + F + H * F + H + 2 * H
    assert blob.size == V * H + P * H + 3 * H + L * per_layer + NL * H + NL
    assert np.array_equal(blob[:H], w["E_w"][0]) and np.array_equal(blob[-NL:], w["b_c"])


def test_windowing_matches_oracle_plan_and_text_roundtrip():
    d = gen.DESCS["base"]
    pool, poff, ptype = gen.entity_pool(500, 9)
    n_tok = np.array([8, 510, 511, 900, 2000])
    rec = gen.make_records(len(n_tok), n_tok, d, pool, poff, ptype, 10)
    win = gen.window_records(rec)
    assert (np.diff(rec["tok_rec_off"]) == n_tok).all()
    # windows follow oracle.decode.window_plan
    wi = 0
    for r, n in enumerate(n_tok):
        for lo, hi, keep in decode.window_plan(int(n)):
            a, b = win["cu_seqlens"][wi], win["cu_seqlens"][wi + 1]
            assert b - a == hi - lo + 2 and win["win_rec"][wi] == r
            assert win["token_ids"][a] == gen.CLS and win["token_ids"][b - 1] == gen.SEP
            assert win["meta"][a, 3] == 0 and win["meta"][b - 1, 3] == 0
            assert win["meta"][a + 1:b - 1, 3].tolist() == [int(k) for k in keep]
            wi += 1
    assert wi == len(win["cu_seqlens"]) - 1
    # decoding the PLANTED labels recovers exactly the planted entity strings, in order
    spans = decode.decode_spans(win["planted_label"], win["meta"])
    assert len(spans) == rec["n_entities"] > 50
    data, off = decode.gather_spans(rec["text"], rec["rec_off"], spans)
    pool_set = {bytes(pool[poff[i]:poff[i + 1]]): int(ptype[i]) for i in range(500)}
    for s, (_, _, _, t) in enumerate(spans):
        e = bytes(data[off[s]:off[s + 1]])
        assert pool_set[e] == t
    # token ids sit in the band of their planted label
    lab = win["planted_label"].astype(int)
    ids = win["token_ids"]
    ent = lab > 0
    assert ((ids[ent] - gen.FIRST_ID) // gen.BAND == lab[ent] - 1).all()
    assert (ids[(lab == 0) & (win["meta"][:, 3] == 1)] >= gen.FIRST_ID + 12 * gen.BAND).all()


def test_zipf_spans_shape():
    data, off, types, key, draws = gen.spans_zipf(2000, 50000, 7, 128, 6, 42)
    lens = np.diff(off)
    assert lens.min() >= 7 and lens.max() <= 128 and key.size == 32
    top = np.bincount(draws).max() / len(draws)
    assert 0.05 < top < 0.35                      # Zipf head
    uniq = {bytes(data[off[i]:off[i + 1]]) for i in range(0, 50000, 7)}
    assert len(uniq) > 300


def test_field_spans_are_the_generated_entity_ranges():
    """NEXT-2 input: gen.field_spans names exactly the entity strings make_records wrote (checked with the oracle's decoder over
    the un-windowed planted labels and against the text itself), with the fixed type in every row."""
    from oracle import decode
    rec = gen.workload_stream(n_records=40, seed=11, n_pool=500)
    sp = gen.field_spans(rec, 3)
    assert sp.dtype == np.int32 and sp.shape == (rec["n_entities"], 4) and (sp[:, 3] == 3).all()
    T = rec["ids"].size
    meta = np.zeros((T, 4), np.int32)
    meta[:, 0] = np.searchsorted(rec["tok_rec_off"], np.arange(T), side="right") - 1
    meta[:, 1], meta[:, 2], meta[:, 3] = rec["char_start"], rec["char_end"], 1
    want = decode.decode_spans(rec["planted_label"].astype(np.int32), meta)
    assert [tuple(r[:3]) for r in sp.tolist()] == [w[:3] for w in want]
    pool, poff, _ = gen.entity_pool(500, 12)
    strings = {pool[poff[i]:poff[i + 1]].tobytes() for i in range(500)}
    for r, cs, ce, _t in sp[:200]:
        base = int(rec["rec_off"][r])
        assert rec["text"][base + cs:base + ce].tobytes() in strings


def test_bench_weight_recipe_covers_both_architectures():
    """bench.py's weight recipe (the deep planted detector) must work for the arch-0 and the arch-1 generator: the arch-1 one
    only takes the shallow triple (`bench.py --workload modern` once died unpacking the longer tuple)."""
    import bench
    for name, d in gen.DESCS.items():
        small = dict(d, layers=1, vocab=min(d["vocab"], 4096))
        w = bench.make_weights_for(small, 7)
        assert len(w["layers"]) == 1 and w["W_c"].shape[0] == small["num_labels"], name
