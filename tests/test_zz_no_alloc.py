"""anon_decode_spans_static: the A9 BIO decode with its scratch in a static device array (no context, no allocation inside
the call; include/anonshield.h).  Checked bit for bit (integer work) against the existing path, anon_decode_spans, on the same
inputs, on two calls in a row that share the static array, and against its size limit.  Collected last on purpose (file name):
the run uses `pytest -x`."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

NT = 4                      # entity types -> 2 * NT + 1 labels
MAX_TOKENS = 1 << 20        # ANON_DECODE_STATIC_MAX_TOKENS


def _stream(rng, T, p_keep, n_rec):
    labels = rng.integers(0, 2 * NT + 1, T).astype(np.int32)
    labels[rng.random(T) < 0.35] = 0
    rec = np.sort(rng.integers(0, n_rec, T)).astype(np.int32)
    cs = np.arange(T, dtype=np.int32) * 5
    meta = np.stack([rec, cs, cs + rng.integers(1, 5, T).astype(np.int32), (rng.random(T) < p_keep).astype(np.int32)], 1)
    return labels, np.ascontiguousarray(meta, np.int32)


@pytest.fixture(scope="module")
def env():
    import torch
    import paper_2606_15650_b200 as P
    if not torch.cuda.is_available():
        pytest.fail("GPU test selected but no CUDA device")
    ctx = P.Context(0, workspace_bytes=64 << 20)
    yield P, torch, ctx
    ctx.close()


def _both(P, torch, ctx, labels, meta, cap):
    dev = "cuda:0"
    d_lab = torch.from_numpy(labels).to(dev)
    d_meta = torch.from_numpy(meta).to(dev)
    out = []
    for static in (False, True):
        spans = torch.full((max(cap, 1), 4), -7, dtype=torch.int32, device=dev)
        num = torch.full((1,), -1, dtype=torch.int32, device=dev)
        if static:
            P.anon_decode_spans_static(0, torch.cuda.current_stream().cuda_stream, d_lab, d_meta, 2 * NT + 1, spans[:cap], num)
            torch.cuda.synchronize()
        else:
            P.anon_decode_spans(ctx, d_lab, d_meta, 2 * NT + 1, spans[:cap], num)
            ctx.sync()                    # the sticky status (CAPACITY on overflow) is read and cleared here
            torch.cuda.synchronize()
        out.append((int(num.item()), spans.cpu().numpy()))
    return out


def test_static_decode_matches_workspace_path_on_two_calls_in_a_row(env):
    P, torch, ctx = env
    rng = np.random.default_rng(2606_15650)
    # a large call first (many tiles + ragged tail), then a smaller one with another keep rate: stale prev_kept / aggregates
    # left in the static array by the first call would show in the second; then the first shape again
    cases = [(300_007, 0.9, 5000), (70_001, 0.3, 900), (300_007, 0.6, 5000), (1, 1.0, 1)]
    for T, p_keep, n_rec in cases:
        labels, meta = _stream(rng, T, p_keep, n_rec)
        (n_ref, s_ref), (n_st, s_st) = _both(P, torch, ctx, labels, meta, T + 1)
        assert n_ref > 0 or T == 1
        assert n_st == n_ref, (T, n_st, n_ref)
        assert np.array_equal(s_st, s_ref), T          # bit-exact, untouched rows (-7) included


def test_static_decode_span_capacity_overflow_reports_total(env):
    P, torch, ctx = env
    rng = np.random.default_rng(7)
    labels, meta = _stream(rng, 50_000, 0.9, 700)
    (n_full, s_full), _ = _both(P, torch, ctx, labels, meta, 50_001)
    cap = n_full // 3
    (n_ref, s_ref), (n_st, s_st) = _both(P, torch, ctx, labels, meta, cap)
    assert n_st == n_ref == n_full and n_st > cap      # the TOTAL count, beyond the capacity
    assert np.array_equal(s_st, s_ref)
    assert np.array_equal(s_st[:cap], s_full[:cap])


def test_static_decode_empty_and_limit(env):
    P, torch, ctx = env
    dev = "cuda:0"
    num = torch.full((1,), -1, dtype=torch.int32, device=dev)
    spans = torch.zeros((4, 4), dtype=torch.int32, device=dev)
    empty_l = torch.zeros(0, dtype=torch.int32, device=dev)
    empty_m = torch.zeros((0, 4), dtype=torch.int32, device=dev)
    P.anon_decode_spans_static(0, 0, empty_l, empty_m, 2 * NT + 1, spans, num)
    torch.cuda.synchronize()
    assert int(num.item()) == 0
    # one token beyond the stated maximum: rejected with CAPACITY before anything is launched
    big_l = torch.zeros(MAX_TOKENS + 1, dtype=torch.int32, device=dev)
    big_m = torch.zeros((MAX_TOKENS + 1, 4), dtype=torch.int32, device=dev)
    num.fill_(-1)
    with pytest.raises(P.AnonError) as ei:
        P.anon_decode_spans_static(0, 0, big_l, big_m, 2 * NT + 1, spans, num)
    assert ei.value.code == P.ERR_CAPACITY
    torch.cuda.synchronize()
    assert int(num.item()) == -1
    with pytest.raises(P.AnonError) as ei:
        P.anon_decode_spans_static(0, 0, big_l[:8], big_m[:8], 2 * NT, spans, num)      # even label count
    assert ei.value.code == P.ERR_UNSUPPORTED
    # exactly the maximum is accepted and agrees with the workspace path
    rng = np.random.default_rng(11)
    labels, meta = _stream(rng, MAX_TOKENS, 0.95, 20_000)
    (n_ref, s_ref), (n_st, s_st) = _both(P, torch, ctx, labels, meta, MAX_TOKENS // 2)
    assert n_st == n_ref and np.array_equal(s_st, s_ref)
