"""GPU parity (through the C ABI) of A11-A13: hash-cache dedup, HMAC-SHA256, pseudonym write-back.
Bar: bit-exact against oracle/crypto.py on the same seeded inputs (BASELINE.json north_star ¶5)."""
import hashlib
import hmac as pyhmac
import os

import numpy as np
import pytest

from harness import gen

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def env():
    import torch
    import paper_2606_15650_b200 as P
    if not torch.cuda.is_available():
        pytest.fail("GPU test selected but no CUDA device: the CUDA path must run, there is no fallback")
    ctx = P.Context(0, workspace_bytes=int(os.environ.get("ANON_TEST_WS", 2 << 30)))
    yield P, torch, ctx
    ctx.close()


def _run_gpu(P, torch, ctx, cache, data, off, types, key, slug_len, names):
    dev = "cuda:0"
    S = off.size - 1
    d_bytes = torch.from_numpy(np.ascontiguousarray(data)).to(dev) if data.size else torch.zeros(16, dtype=torch.uint8, device=dev)
    d_off = torch.from_numpy(np.ascontiguousarray(off, np.int64)).to(dev)
    d_type = None if types is None else torch.from_numpy(np.ascontiguousarray(types, np.uint8)).to(dev)
    cap = S * (3 + max(len(n) for n in names) + slug_len) + 16
    out = torch.zeros(cap, dtype=torch.uint8, device=dev)
    out_off = torch.zeros(S + 1, dtype=torch.int64, device=dev)
    hit = torch.zeros(max(S, 1), dtype=torch.uint8, device=dev)
    uid = torch.zeros(max(S, 1), dtype=torch.int64, device=dev)
    dig = torch.zeros((max(S, 1), 32), dtype=torch.uint8, device=dev)
    P.anon_pseudonymize(ctx, cache, d_bytes, d_off, d_type, key, slug_len, names, out, out_off, hit, uid, dig)
    assert ctx.sync() == 0
    oo = out_off.cpu().numpy()
    return {"out_tokens": out.cpu().numpy()[:oo[S]], "out_offsets": oo, "hit": hit.cpu().numpy()[:S],
            "uid": uid.cpu().numpy()[:S], "digests": dig.cpu().numpy()[:S]}


def _assert_same(got, want):
    for k in ("out_offsets", "hit", "uid", "digests", "out_tokens"):
        assert got[k].shape == want[k].shape, k
        assert np.array_equal(got[k], want[k]), k


def test_config1_spans_bit_exact_and_slug_sweep(env):
    """BASELINE.json configs[0]: 1,000 ASCII spans of 4-64 bytes, 30 % duplicates, 32-byte key."""
    P, torch, ctx = env
    from oracle import crypto
    data, off, types, key = gen.spans_config1()
    for slug_len in (10, 0, 1, 63, 64):
        oc = crypto.Cache()
        want = oc.pseudonymize(data, off, types, key.tobytes(), slug_len, gen.TYPE_NAMES_4)
        gc = P.Cache(ctx, 4096, 1 << 20)
        got = _run_gpu(P, torch, ctx, gc, data, off, types, key.tobytes(), slug_len, gen.TYPE_NAMES_4)
        _assert_same(got, want)
        assert gc.stats() == oc.stats()
        # P:L44 surface form and an independent hashlib check of span 0
        tok0 = bytes(got["out_tokens"][got["out_offsets"][0]:got["out_offsets"][1]]).decode()
        e0 = bytes(data[off[0]:off[1]])
        assert tok0 == "[%s_%s]" % (gen.TYPE_NAMES_4[types[0]], pyhmac.new(key.tobytes(), e0, hashlib.sha256).hexdigest()[:slug_len])
        # cache export row: entity bytes + full digest by uid
        eb, dg = gc.entry(int(got["uid"][0]))
        assert eb == e0 and dg == pyhmac.new(key.tobytes(), e0, hashlib.sha256).digest()
        gc.close(); oc.close()


def test_referential_integrity_across_calls_and_keys(env):
    """same (key, entity) -> same pseudonym in any batch/position; splitting a call changes nothing."""
    P, torch, ctx = env
    from oracle import crypto
    data, off, types, key = gen.spans_config1()
    oc, gc = crypto.Cache(), P.Cache(ctx, 4096, 1 << 20)
    cuts = [0, 1, 137, 138, 600, 1000]
    for a, b in zip(cuts[:-1], cuts[1:]):
        sub_off = off[a:b + 1] - off[a]
        sub = data[off[a]:off[b]]
        want = oc.pseudonymize(sub, sub_off, types[a:b], key.tobytes(), 10, gen.TYPE_NAMES_4)
        got = _run_gpu(P, torch, ctx, gc, sub, sub_off, types[a:b], key.tobytes(), 10, gen.TYPE_NAMES_4)
        _assert_same(got, want)
    # second pass over everything: all hits, same tokens
    want = oc.pseudonymize(data, off, types, key.tobytes(), 10, gen.TYPE_NAMES_4)
    got = _run_gpu(P, torch, ctx, gc, data, off, types, key.tobytes(), 10, gen.TYPE_NAMES_4)
    _assert_same(got, want)
    assert got["hit"].all() and gc.stats() == oc.stats()
    # another key on the same cache is refused; on a fresh cache it gives different digests
    with pytest.raises(P.AnonError) as ei:
        _run_gpu(P, torch, ctx, gc, data, off, types, b"another key", 10, gen.TYPE_NAMES_4)
    assert ei.value.code == -4
    g2 = P.Cache(ctx, 4096, 1 << 20)
    other = _run_gpu(P, torch, ctx, g2, data, off, types, b"another key", 10, gen.TYPE_NAMES_4)
    assert not (other["digests"] == got["digests"]).all(axis=1).any()
    gc.close(); g2.close(); oc.close()


def test_edge_cases(env):
    """Empty call, zero-length messages, every SHA padding boundary, long keys, NULL type array."""
    P, torch, ctx = env
    from oracle import crypto
    rng = np.random.default_rng(5)
    lens = [0, 1, 3, 4, 5, 55, 56, 57, 63, 64, 65, 119, 120, 121, 127, 128, 183, 184, 300, 0, 55, 64]
    off = np.zeros(len(lens) + 1, np.int64)
    off[1:] = np.cumsum(lens)
    data = rng.integers(0, 256, int(off[-1])).astype(np.uint8)
    for key in (b"", b"k", bytes(range(64)), bytes(range(65)), bytes(rng.integers(0, 256, 131).astype(np.uint8))):
        oc, gc = crypto.Cache(), P.Cache(ctx, 64, 4096)
        want = oc.pseudonymize(data, off, None, key, 64, ["T"])
        got = _run_gpu(P, torch, ctx, gc, data, off, None, key, 64, ["T"])
        _assert_same(got, want)
        for i, n in enumerate(lens):   # independent of the oracle: Python's hmac
            assert bytes(got["digests"][i]) == pyhmac.new(key, bytes(data[off[i]:off[i + 1]]), hashlib.sha256).digest()
        gc.close(); oc.close()
    gc = P.Cache(ctx, 64, 4096)
    got = _run_gpu(P, torch, ctx, gc, np.zeros(0, np.uint8), np.zeros(1, np.int64), None, b"k", 10, ["T"])
    assert got["out_tokens"].size == 0 and got["out_offsets"].tolist() == [0]
    gc.close()


def test_capacity_errors_leave_cache_unchanged(env):
    P, torch, ctx = env
    from oracle import crypto
    data, off, types, key = gen.spans_config1()
    gc = P.Cache(ctx, 100, 1 << 20)         # 700 unique do not fit
    with pytest.raises(P.AnonError) as ei:
        _run_gpu(P, torch, ctx, gc, data, off, types, key.tobytes(), 10, gen.TYPE_NAMES_4)
    assert ei.value.code == -3 and gc.stats()["n_unique"] == 0
    # the same cache still works, bit-exact, for a part that fits
    oc = crypto.Cache()
    n = 90
    want = oc.pseudonymize(data[:off[n]], off[:n + 1], types[:n], key.tobytes(), 10, gen.TYPE_NAMES_4)
    got = _run_gpu(P, torch, ctx, gc, data[:off[n]], off[:n + 1], types[:n], key.tobytes(), 10, gen.TYPE_NAMES_4)
    _assert_same(got, want)
    gc.close(); oc.close()
    g2 = P.Cache(ctx, 4096, 100)            # arena too small
    with pytest.raises(P.AnonError) as ei:
        _run_gpu(P, torch, ctx, g2, data, off, types, key.tobytes(), 10, gen.TYPE_NAMES_4)
    assert ei.value.code == -3
    g2.close()


def test_hmac_only_kernel_matches_oracle(env):
    P, torch, ctx = env
    from oracle import crypto
    data, off, _t, key, _d = gen.spans_zipf(5000, 200000, 7, 128, 6, gen.SEED_BASE + 55)
    want = crypto.hmac_batch(key.tobytes(), data, off)
    dev = "cuda:0"
    dig = torch.zeros((off.size - 1, 32), dtype=torch.uint8, device=dev)
    P.anon_hmac_spans(ctx, torch.from_numpy(data).to(dev), torch.from_numpy(off).to(dev), key.tobytes(), dig)
    assert ctx.sync() == 0
    assert np.array_equal(dig.cpu().numpy(), want)


@pytest.mark.parametrize("n_unique,n_draws", [(200_000, 5_000_000)])
def test_zipf_stress_shape_bit_exact(env, n_unique, n_draws):
    """BASELINE.json configs[4] shape (7-128 byte spans, Zipf(1.1), heavy head contention) at 1/10 scale,
    full oracle comparison; the full 50 M run is `bench.py --workload pseudonym` with sampled checks."""
    P, torch, ctx = env
    from oracle import crypto
    data, off, types, key, _d = gen.spans_zipf(n_unique, n_draws, 7, 128, 6, gen.SEED_BASE + 5)
    oc = crypto.Cache(1 << 20)
    want = oc.pseudonymize(data, off, types, key.tobytes(), 10, gen.TYPE_NAMES_6)
    gc = P.Cache(ctx, n_unique, int(off[-1] // 4) + (1 << 20))
    got = _run_gpu(P, torch, ctx, gc, data, off, types, key.tobytes(), 10, gen.TYPE_NAMES_6)
    _assert_same(got, want)
    assert gc.stats() == oc.stats()
    gc.close(); oc.close()


def test_cache_export_is_the_mapping_table_and_resumes(env):
    """P:L52 hand-off: the exported rows are (entity, HMAC-SHA256(key, entity)) in first-occurrence order -- checked
    against Python's own hmac / dict, not the oracle -- and re-inserting them into a fresh cache reproduces uids and
    digests, after which the original spans are all hits (checkpoint / resume)."""
    P, torch, ctx = env
    data, off, types, key = gen.spans_config1()
    kb = key.tobytes()
    gc = P.Cache(ctx, 4096, 1 << 20)
    first = _run_gpu(P, torch, ctx, gc, data, off, types, kb, 10, gen.TYPE_NAMES_4)
    ebytes, eoff, edig = gc.export()
    seen = {}
    for i in range(off.size - 1):
        seen.setdefault(bytes(data[off[i]:off[i + 1]]), len(seen))
    ents = sorted(seen, key=seen.get)
    assert eoff.size - 1 == len(ents) == edig.shape[0]
    for u, e in enumerate(ents):
        assert bytes(ebytes[eoff[u]:eoff[u + 1]]) == e
        assert bytes(edig[u]) == pyhmac.new(kb, e, hashlib.sha256).digest()
    gc.close()
    # resume: a fresh cache fed with the exported entities, then the original spans
    g2 = P.Cache(ctx, 4096, 1 << 20)
    r = _run_gpu(P, torch, ctx, g2, ebytes, eoff, None, kb, 10, gen.TYPE_NAMES_4)
    assert not r["hit"].any() and np.array_equal(r["uid"], np.arange(len(ents))) and np.array_equal(r["digests"], edig)
    again = _run_gpu(P, torch, ctx, g2, data, off, types, kb, 10, gen.TYPE_NAMES_4)
    assert again["hit"].all() and np.array_equal(again["uid"], first["uid"]) and np.array_equal(again["out_tokens"], first["out_tokens"])
    g2.close()


def test_bounded_cache_eviction_matches_oracle(env):
    """NEXT-5 (reading D21): a Zipf span stream in 12 calls with an eviction after most of them; hit flags, uids and digests
    of every call, the surviving entries in uid order and the counters equal oracle/cache_lru.py."""
    P, torch, ctx = env
    from oracle import cache_lru
    key = bytes(range(40, 72))
    pool, poff, _t = gen.entity_pool(3000, 17)
    ents = [pool[poff[i]:poff[i + 1]].tobytes() for i in range(3000)]
    rng = np.random.default_rng(12)
    oc = cache_lru.LruCache(key)
    gc = P.Cache(ctx, 4096, 1 << 20)
    with pytest.raises(P.AnonError) as ei:                      # eviction needs recency tracking
        gc.evict(10)
    assert ei.value.code == -2
    gc.track_use()
    keeps = [None, 900, 900, None, 300, 300, 2000, 1, 50, 0, None, 40]
    for step, keep in enumerate(keeps):
        draws = np.minimum(rng.zipf(1.15, 4000) - 1, 2999) if step != 7 else np.arange(5)
        spans = [ents[int(v)] for v in draws]
        data = np.frombuffer(b"".join(spans), np.uint8).copy()
        off = np.zeros(len(spans) + 1, np.int64); off[1:] = np.cumsum([len(s) for s in spans])
        got = _run_gpu(P, torch, ctx, gc, data, off, None, key, 10, gen.TYPE_NAMES_4)
        hit, uid, dig = oc.pseudonymize(spans)
        assert np.array_equal(got["hit"], np.asarray(hit, np.uint8)), step
        assert np.array_equal(got["uid"], np.asarray(uid, np.int64)), step
        assert np.array_equal(got["digests"], np.frombuffer(b"".join(dig), np.uint8).reshape(-1, 32)), step
        if keep is not None:
            assert gc.evict(keep) == oc.evict(keep), step
        bytes_, offs, digs = gc.export()
        want = oc.export()
        assert offs.size - 1 == len(want), step
        assert [bytes_[offs[i]:offs[i + 1]].tobytes() for i in range(len(want))] == [e for e, _d in want], step
        assert digs.tobytes() == b"".join(d for _e, d in want), step
        st = gc.stats()
        assert (st["n_unique"], st["n_lookups"], st["n_hits"]) == (len(want), oc.n_lookups, oc.n_hits), step
    gc.close()


def test_buffers_at_odd_byte_addresses_and_misaligned_digests(env):
    """ABI alignment rules (include/anonshield.h, anon_pseudonymize): span bytes and the token buffer may sit at ANY byte address
    (sub-buffers of a larger allocation: offsets 1, 2, 3 from a 16-byte boundary), results stay bit-exact; a digest buffer that
    is not 16-byte aligned is rejected with INVALID_ARG instead of faulting."""
    from oracle import crypto
    P, torch, ctx = env
    dev = "cuda:0"
    data, off, types, key = gen.spans_config1()
    S = off.size - 1
    oc = crypto.Cache()
    want = oc.pseudonymize(data, off, types, key.tobytes(), 10, gen.TYPE_NAMES_4)
    oc.close()
    for shift in (1, 2, 3, 7):
        cache = P.Cache(ctx, 4096, 1 << 20)
        big_in = torch.zeros(data.size + 64, dtype=torch.uint8, device=dev)
        big_in[shift:shift + data.size] = torch.from_numpy(data).to(dev)
        big_out = torch.zeros(S * 32 + 64, dtype=torch.uint8, device=dev)
        out = big_out[shift:]
        assert out.data_ptr() % 4 == shift % 4
        out_off = torch.zeros(S + 1, dtype=torch.int64, device=dev)
        hit = torch.zeros(S + 8, dtype=torch.uint8, device=dev)[shift:shift + S]
        P.anon_pseudonymize(ctx, cache, big_in[shift:shift + data.size], torch.from_numpy(off).to(dev), torch.from_numpy(types).to(dev),
                            key.tobytes(), 10, gen.TYPE_NAMES_4, out, out_off, hit)
        assert ctx.sync() == 0
        oo = out_off.cpu().numpy()
        assert np.array_equal(oo, want["out_offsets"])
        assert np.array_equal(out.cpu().numpy()[:oo[S]], want["out_tokens"])
        assert np.array_equal(hit.cpu().numpy(), want["hit"])
        assert int(big_out[:shift].sum()) == 0 and int(big_out[shift + oo[S]:].sum()) == 0     # nothing outside the token range
        cache.close()
    cache = P.Cache(ctx, 4096, 1 << 20)
    dig = torch.zeros(S * 32 + 16, dtype=torch.uint8, device=dev)[4:]
    out = torch.zeros(S * 32, dtype=torch.uint8, device=dev)
    with pytest.raises(P.AnonError) as e:
        P.anon_pseudonymize(ctx, cache, torch.from_numpy(data).to(dev), torch.from_numpy(off).to(dev), None, key.tobytes(), 10,
                            gen.TYPE_NAMES_4, out, torch.zeros(S + 1, dtype=torch.int64, device=dev), None, None, dig)
    assert e.value.code == P.ERR_INVALID_ARG
    with pytest.raises(P.AnonError) as e:
        P.anon_hmac_spans(ctx, torch.from_numpy(data).to(dev), torch.from_numpy(off).to(dev), key.tobytes(), dig)
    assert e.value.code == P.ERR_INVALID_ARG
    assert cache.stats()["n_unique"] == 0
    cache.close()


def test_cache_protocol_is_order_deterministic(env):
    """The CAS + atomicMin slot protocol must give the sequential definition's answer whatever the thread schedule: the same
    span list run 5 times on fresh caches gives identical hit / uid arrays (= the oracle's), and a shuffled copy of the list
    gives the oracle's answer for THAT order (uids follow first occurrence in the new order) with the same set of digests."""
    from oracle import crypto
    P, torch, ctx = env
    data, off, types, key, draws = gen.spans_zipf(3000, 200_000, 7, 128, 6, 77)
    kb = key.tobytes()
    oc = crypto.Cache(1 << 14)
    want = oc.pseudonymize(data, off, types, kb, 10, gen.TYPE_NAMES_6)
    oc.close()
    for _ in range(5):
        cache = P.Cache(ctx, 4096, 1 << 20)
        got = _run_gpu(P, torch, ctx, cache, data, off, types, kb, 10, gen.TYPE_NAMES_6)
        cache.close()
        _assert_same(got, want)
    perm = np.random.default_rng(3).permutation(off.size - 1)
    pool, poff = gen.ascii_pool(3000, 7, 128, 77 + 1000)
    data2, off2 = gen.expand_csr(pool, poff, draws[perm])
    oc = crypto.Cache(1 << 14)
    want2 = oc.pseudonymize(data2, off2, types[perm], kb, 10, gen.TYPE_NAMES_6)
    oc.close()
    cache = P.Cache(ctx, 4096, 1 << 20)
    got2 = _run_gpu(P, torch, ctx, cache, data2, off2, types[perm], kb, 10, gen.TYPE_NAMES_6)
    cache.close()
    _assert_same(got2, want2)
    assert np.array_equal(got2["digests"], got["digests"][perm])            # a pseudonym never depends on the order
