"""Pins of oracle/cache_lru.py (NEXT-5, reading D21)."""
import collections
import hashlib
import hmac

import numpy as np

from oracle import cache_lru


def test_hand_worked_trace():
    c = cache_lru.LruCache(b"k")
    assert c.pseudonymize([b"a", b"b", b"a", b"c"])[:2] == ([0, 0, 1, 0], [0, 1, 0, 2])      # call 1 stamps a, b, c
    assert c.pseudonymize([b"b", b"d"])[:2] == ([1, 0], [1, 3])                              # call 2 stamps b, d
    assert c.pseudonymize([b"a"])[:2] == ([1], [0])                                          # call 3 stamps a
    # stamps: a 3, b 2, c 1, d 2.  keep 3 drops c; keep 2 keeps a (3) and, of the two entries stamped 2, the lower uid b
    assert c.evict(3) == 1 and [e for e, _d in c.export()] == [b"a", b"b", b"d"]
    assert c.evict(2) == 1 and [e for e, _d in c.export()] == [b"a", b"b"]
    assert c.evict(5) == 0
    hit, uid, dig = c.pseudonymize([b"d", b"b", b"c"])                                       # d and c are misses again
    assert (hit, uid) == ([0, 1, 0], [2, 1, 3])
    assert dig[0] == hmac.new(b"k", b"d", hashlib.sha256).digest()                           # same pseudonym as before
    assert (c.n_lookups, c.n_hits) == (10, 4)
    assert c.evict(0) == 4 and c.export() == []


def test_single_span_calls_are_a_textbook_lru():
    """One span per call and evict(C) after every call: the hit / miss sequence of an LRU of capacity C, here checked against
    collections.OrderedDict (move_to_end / popitem), an independent structure."""
    rng = np.random.default_rng(4)
    for cap in (1, 3, 8):
        c = cache_lru.LruCache(b"key")
        ref = collections.OrderedDict()
        for x in rng.zipf(1.3, 600) % 40:
            e = b"e%d" % x
            hit = c.pseudonymize([e])[0][0]
            c.evict(cap)
            want = 1 if e in ref else 0
            ref[e] = True
            ref.move_to_end(e)
            if len(ref) > cap:
                ref.popitem(last=False)
            assert hit == want
            assert sorted(k for k, _d in c.export()) == sorted(ref)


def test_pseudonyms_do_not_depend_on_evictions():
    rng = np.random.default_rng(5)
    a, b = cache_lru.LruCache(b"key"), cache_lru.LruCache(b"key")
    for step in range(30):
        spans = [b"ent%d" % v for v in rng.zipf(1.2, 50) % 200]
        da = a.pseudonymize(spans)[2]
        db = b.pseudonymize(spans)[2]
        assert da == db
        b.evict(20)
        assert len(b.export()) <= 20
    assert a.n_lookups == b.n_lookups and a.n_hits > b.n_hits
