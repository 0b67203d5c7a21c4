"""GPU parity (through the C ABI) of A9 BIO decode + compaction and A10 span byte gather.
Bar: span offsets bit-exact against oracle/decode.py (BASELINE.json north_star ¶5)."""
import os

import numpy as np
import pytest

from harness import gen
from test_oracle_decode import _parse_case

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def env():
    import torch
    import paper_2606_15650_b200 as P
    if not torch.cuda.is_available():
        pytest.fail("GPU test selected but no CUDA device")
    ctx = P.Context(0, workspace_bytes=512 << 20)
    yield P, torch, ctx
    ctx.close()


def _gpu_decode(P, torch, ctx, labels, meta, num_labels, cap=None):
    dev = "cuda:0"
    T = len(labels)
    cap = T + 1 if cap is None else cap
    d_lab = torch.from_numpy(np.ascontiguousarray(labels, np.int32)).to(dev) if T else torch.zeros(1, dtype=torch.int32, device=dev)[:0]
    d_meta = torch.from_numpy(np.ascontiguousarray(meta, np.int32).reshape(-1, 4)).to(dev) if T else torch.zeros((0, 4), dtype=torch.int32, device=dev)
    spans = torch.full((max(cap, 1), 4), -7, dtype=torch.int32, device=dev)
    num = torch.zeros(1, dtype=torch.int32, device=dev)
    P.anon_decode_spans(ctx, d_lab, d_meta, num_labels, spans[:cap], num)
    rc = ctx.sync()
    n = int(num.item())
    return rc, n, spans.cpu().numpy()[:min(n, cap)]


def test_hand_worked_cases_on_gpu(env, golden_dir):
    P, torch, ctx = env
    with open(os.path.join(golden_dir, "bio_cases.txt")) as f:
        for line in f:
            if not line.strip() or line.startswith("#"):
                continue
            labels, meta, want = _parse_case(line)
            rc, n, spans = _gpu_decode(P, torch, ctx, labels, meta, 5)
            assert rc == 0 and n == len(want), line
            assert [tuple(int(v) for v in s) for s in spans] == want, line


def _random_stream(rng, T, nt, p_keep, n_rec):
    labels = rng.integers(0, 2 * nt + 1, T).astype(np.int32)
    labels[rng.random(T) < 0.35] = 0
    rec = np.sort(rng.integers(0, n_rec, T)).astype(np.int32)
    cs = np.arange(T, dtype=np.int32) * 5
    meta = np.stack([rec, cs, cs + rng.integers(1, 5, T).astype(np.int32), (rng.random(T) < p_keep).astype(np.int32)], 1)
    return labels, meta


@pytest.mark.parametrize("T,p_keep", [(1, 1.0), (31, 0.9), (2048, 0.8), (2049, 0.5), (100_003, 0.97), (300_000, 0.02)])
def test_random_streams_match_oracle(env, T, p_keep):
    """Several scan tiles plus a ragged tail; sparse keep flags exercise long transparent runs."""
    P, torch, ctx = env
    from oracle import decode
    rng = np.random.default_rng(T)
    labels, meta = _random_stream(rng, T, 6, p_keep, max(1, T // 300))
    want = decode.decode_spans(labels, meta)
    rc, n, spans = _gpu_decode(P, torch, ctx, labels, meta, 13)
    assert rc == 0 and n == len(want)
    assert np.array_equal(spans, np.asarray(want, np.int32).reshape(-1, 4))


def test_empty_none_kept_and_capacity(env):
    P, torch, ctx = env
    rc, n, _ = _gpu_decode(P, torch, ctx, np.zeros(0, np.int32), np.zeros((0, 4), np.int32), 13)
    assert rc == 0 and n == 0
    rng = np.random.default_rng(1)
    labels, meta = _random_stream(rng, 5000, 6, 1.0, 3)
    meta0 = meta.copy(); meta0[:, 3] = 0
    rc, n, _ = _gpu_decode(P, torch, ctx, labels, meta0, 13)
    assert rc == 0 and n == 0
    from oracle import decode
    want = decode.decode_spans(labels, meta)
    rc, n, spans = _gpu_decode(P, torch, ctx, labels, meta, 13, cap=10)
    assert rc == -3 and n == len(want)                       # ANON_ERR_CAPACITY latched, needed count reported
    assert np.array_equal(spans, np.asarray(want[:10], np.int32))
    assert ctx.sync() == 0                                   # sticky status was cleared


def test_windowed_records_decode_and_gather(env):
    """Planted labels on windowed records (510+2 tokens, 128 overlap, midpoint ownership): spans cross window
    boundaries; the gathered bytes are exactly the planted entity strings."""
    P, torch, ctx = env
    from oracle import decode
    d = gen.DESCS["base"]
    pool, poff, ptype = gen.entity_pool(800, 21)
    n_tok = np.array([8, 510, 511, 893, 2000, 3000, 40, 1275])
    rec = gen.make_records(len(n_tok), n_tok, d, pool, poff, ptype, 22)
    win = gen.window_records(rec)
    want = decode.decode_spans(win["planted_label"], win["meta"])
    rc, n, spans = _gpu_decode(P, torch, ctx, win["planted_label"].astype(np.int32), win["meta"], 13)
    assert rc == 0 and n == len(want) == rec["n_entities"]
    assert np.array_equal(spans, np.asarray(want, np.int32))
    wb, wo = decode.gather_spans(rec["text"], rec["rec_off"], want)
    dev = "cuda:0"
    d_sp = torch.from_numpy(spans).to(dev)
    sb = torch.zeros(int(wo[-1]) + 16, dtype=torch.uint8, device=dev)
    so = torch.zeros(n + 1, dtype=torch.int64, device=dev)
    stype = torch.zeros(n, dtype=torch.uint8, device=dev)
    P.anon_gather_spans(ctx, torch.from_numpy(rec["text"]).to(dev), torch.from_numpy(rec["rec_off"]).to(dev), d_sp, n,
                        sb, so, stype)
    assert ctx.sync() == 0
    assert np.array_equal(so.cpu().numpy(), wo)
    assert np.array_equal(sb.cpu().numpy()[:wo[-1]], wb)
    assert np.array_equal(stype.cpu().numpy(), spans[:, 3].astype(np.uint8))
    # capacity: one byte short
    sb2 = torch.zeros(int(wo[-1]) - 1, dtype=torch.uint8, device=dev)
    P.anon_gather_spans(ctx, torch.from_numpy(rec["text"]).to(dev), torch.from_numpy(rec["rec_off"]).to(dev), d_sp, n,
                        sb2, so, None)
    assert ctx.sync() == -3


def test_splice_records_matches_oracle(env):
    """NEXT-1: every record rewritten with its spans replaced by their pseudonym tokens, bit-exact against
    oracle/decode.splice_records; tokens longer and shorter than the spans, records without spans, S = 0, capacity."""
    P, torch, ctx = env
    from oracle import crypto, decode
    dev = "cuda:0"
    d = dict(gen.DESCS["tiny"])
    pool, poff, ptype = gen.entity_pool(64, 3)
    n_tok = np.array([40, 700, 90, 8, 1300, 16, 300, 8, 8, 64], np.int64)
    rec = gen.make_records(len(n_tok), n_tok, d, pool, poff, ptype % 4, 5, entity_rate=1.0 / 12)
    win = gen.window_records(rec)
    spans = decode.decode_spans(win["planted_label"].astype(np.int32), win["meta"])
    assert len(spans) > 100
    sb, so = decode.gather_spans(rec["text"], rec["rec_off"], spans)
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(dev)
    for slug_len in (10, 0, 64):
        oc = crypto.Cache()
        ps = oc.pseudonymize(sb, so, np.asarray([s[3] for s in spans], np.uint8), bytes(range(32)), slug_len, gen.TYPE_NAMES_4)
        oc.close()
        want, want_off = decode.splice_records(rec["text"], rec["rec_off"], spans, ps["out_tokens"], ps["out_offsets"])
        new_text = torch.full((want.size + 64,), 0xEE, dtype=torch.uint8, device=dev)
        new_off = torch.zeros(len(n_tok) + 1, dtype=torch.int64, device=dev)
        P.anon_splice_records(ctx, t(rec["text"]), t(rec["rec_off"]), t(np.asarray(spans, np.int32).reshape(-1, 4)), len(spans),
                              t(ps["out_tokens"]) if ps["out_tokens"].size else torch.zeros(16, dtype=torch.uint8, device=dev),
                              t(ps["out_offsets"]), new_text, new_off)
        assert ctx.sync() == 0
        assert np.array_equal(new_off.cpu().numpy(), want_off)
        got = new_text.cpu().numpy()
        assert np.array_equal(got[:want.size], want) and (got[want.size:] == 0xEE).all()
    # no spans: identity
    new_text = torch.zeros(rec["text"].size, dtype=torch.uint8, device=dev)
    new_off = torch.zeros(len(n_tok) + 1, dtype=torch.int64, device=dev)
    P.anon_splice_records(ctx, t(rec["text"]), t(rec["rec_off"]), torch.zeros((1, 4), dtype=torch.int32, device=dev), 0,
                          torch.zeros(16, dtype=torch.uint8, device=dev), torch.zeros(1, dtype=torch.int64, device=dev), new_text, new_off)
    assert ctx.sync() == 0
    assert np.array_equal(new_text.cpu().numpy(), rec["text"]) and np.array_equal(new_off.cpu().numpy(), rec["rec_off"])
    # capacity too small: latched, nothing written past the end
    small = torch.full((want.size - 100,), 0xEE, dtype=torch.uint8, device=dev)
    P.anon_splice_records(ctx, t(rec["text"]), t(rec["rec_off"]), t(np.asarray(spans, np.int32).reshape(-1, 4)), len(spans),
                          t(ps["out_tokens"]), t(ps["out_offsets"]), small, new_off)
    assert ctx.sync() == -3


def test_splice_edge_cases_and_unaligned_buffers(env):
    """Hand-built records: a span covering a whole record, spans that touch (no gap between them), a span at offset 0 and one
    ending at the record's end, an empty record, an empty token; text / token / output buffers at odd byte addresses."""
    P, torch, ctx = env
    from oracle import decode
    dev = "cuda:0"
    recs = [b"ABCDEFGHIJ", b"", b"0123456789abcdefghijklmnopqrstuvwxyz" * 40, b"xy", b"tail-span-here"]
    text = np.frombuffer(b"".join(recs), np.uint8).copy()
    ro = np.zeros(len(recs) + 1, np.int64)
    ro[1:] = np.cumsum([len(r) for r in recs])
    spans = [(0, 0, 10, 0),                                  # the whole record
             (2, 0, 3, 1), (2, 3, 7, 2), (2, 7, 8, 0),       # at offset 0, touching each other
             (2, 500, 530, 1), (2, 1430, 1440, 3),           # ... the last one ends at the record's end
             (3, 1, 2, 0), (4, 5, 14, 2)]
    toks = [b"[T0_aaaaaaaaaaaaaaaaaaaaaaaaaaaaaaaa]", b"", b"[X]", b"[LONGER_THAN_THE_SPAN]", b"[s]", b"[END]", b"[ONE_BYTE_SPAN]", b"[t]"]
    tok = np.frombuffer(b"".join(toks), np.uint8).copy()
    to = np.zeros(len(toks) + 1, np.int64)
    to[1:] = np.cumsum([len(x) for x in toks])
    want, want_off = decode.splice_records(text, ro, spans, tok, to)
    # independent check of the oracle on this case: plain Python string surgery
    exp = []
    for r, body in enumerate(recs):
        out, cur = b"", 0
        for (rr, cs, ce, _t), tk in zip(spans, toks):
            if rr == r:
                out += body[cur:cs] + tk
                cur = ce
        exp.append(out + body[cur:])
    assert want.tobytes() == b"".join(exp)
    for shift in (0, 1, 5, 13):
        big_text = torch.zeros(text.size + 32, dtype=torch.uint8, device=dev)
        big_text[shift:shift + text.size] = torch.from_numpy(text).to(dev)
        big_tok = torch.zeros(tok.size + 32, dtype=torch.uint8, device=dev)
        big_tok[(shift + 2):(shift + 2) + tok.size] = torch.from_numpy(tok).to(dev)
        big_out = torch.full((want.size + 64,), 0xEE, dtype=torch.uint8, device=dev)
        out = big_out[shift:shift + want.size + 8]
        new_off = torch.zeros(len(recs) + 1, dtype=torch.int64, device=dev)
        P.anon_splice_records(ctx, big_text[shift:shift + text.size], torch.from_numpy(ro).to(dev),
                              torch.from_numpy(np.asarray(spans, np.int32)).to(dev), len(spans), big_tok[(shift + 2):(shift + 2) + tok.size],
                              torch.from_numpy(to).to(dev), out, new_off)
        assert ctx.sync() == 0
        assert np.array_equal(new_off.cpu().numpy(), want_off)
        got = big_out.cpu().numpy()
        assert np.array_equal(got[shift:shift + want.size], want)
        assert (got[:shift] == 0xEE).all() and (got[shift + want.size:] == 0xEE).all()
