"""Pins for oracle/anon_oracle.c (SHA-256, HMAC, dedup, write-back) -- CPU only."""
import hashlib
import hmac as pyhmac
import os
import re

import numpy as np
import pytest

from oracle import crypto


def _spec(s):
    kind, _, rest = s.partition(":")
    if kind == "lit":
        return rest.replace("_", " ").encode()
    if kind == "hex":
        return bytes.fromhex(rest)
    if kind == "rep":
        b, n = rest.split(":")
        return bytes.fromhex(b) * int(n)
    raise ValueError(s)


def _lines(path):
    with open(path) as f:
        return [l.rstrip("\n") for l in f if l.strip() and not l.startswith("#")]


def test_sha256_fips_vectors(golden_dir):
    for line in _lines(os.path.join(golden_dir, "sha256_vectors.txt")):
        spec, _, digest = line.rpartition(" ")
        if spec.startswith("rep:"):
            ch, n = spec[4:].split(":")
            msg = ch.encode() * int(n)
        else:
            msg = spec[4:].encode()
        assert crypto.sha256(msg).hex() == digest, spec[:40]


def test_hmac_rfc4231_vectors(golden_dir):
    for line in _lines(os.path.join(golden_dir, "hmac_vectors.txt")):
        k, m, digest = line.split(" ")
        assert crypto.hmac_sha256(_spec(k), _spec(m)).hex() == digest, line[:40]


def test_constants_from_roots(golden_dir):
    k, h = crypto.sha256_constants()
    for line in _lines(os.path.join(golden_dir, "sha256_constants.txt")):
        which, idx, val = line.split()
        got = (k if which == "K" else h)[int(idx)]
        assert int(got) == int(val, 16)
    # independent derivation with Python big integers: floor(frac(p^(1/3)) * 2^32)
    primes = [p for p in range(2, 400) if all(p % d for d in range(2, int(p ** 0.5) + 1))][:64]

    def iroot(n, r):
        lo, hi = 0, 1 << 80
        while hi - lo > 1:
            mid = (lo + hi) // 2
            if mid ** r <= n:
                lo = mid
            else:
                hi = mid
        return lo
    for i, p in enumerate(primes):
        assert int(k[i]) == iroot(p << 96, 3) & 0xFFFFFFFF
    for i, p in enumerate(primes[:8]):
        assert int(h[i]) == iroot(p << 64, 2) & 0xFFFFFFFF


PAD_LENGTHS = [0, 1, 3, 54, 55, 56, 57, 63, 64, 65, 118, 119, 120, 121, 127, 128, 129, 183, 184, 1000]


def test_sha256_vs_hashlib_every_padding_boundary():
    g = np.random.default_rng(7)
    for n in PAD_LENGTHS:
        m = g.integers(0, 256, n).astype(np.uint8).tobytes()
        assert crypto.sha256(m) == hashlib.sha256(m).digest(), n


def test_hmac_vs_python_hmac_key_and_message_lengths():
    g = np.random.default_rng(8)
    for kl in [0, 1, 32, 63, 64, 65, 131]:
        key = g.integers(0, 256, kl).astype(np.uint8).tobytes()
        for n in PAD_LENGTHS:
            m = g.integers(0, 256, n).astype(np.uint8).tobytes()
            assert crypto.hmac_sha256(key, m) == pyhmac.new(key, m, hashlib.sha256).digest(), (kl, n)


def test_hmac_is_the_two_hash_definition():
    key, m = b"k" * 40, b"some entity"
    kp = key + b"\0" * 24
    inner = hashlib.sha256(bytes(x ^ 0x36 for x in kp) + m).digest()
    want = hashlib.sha256(bytes(x ^ 0x5c for x in kp) + inner).digest()
    assert crypto.hmac_sha256(key, m) == want


def _csr(strs):
    off = np.zeros(len(strs) + 1, np.int64)
    off[1:] = np.cumsum([len(s) for s in strs])
    return np.frombuffer(b"".join(strs), np.uint8), off


def _random_spans(g, n, n_unique, lo=0, hi=40):
    pool = list({bytes(g.integers(0x21, 0x7F, int(g.integers(lo, hi + 1))).astype(np.uint8)) for _ in range(n_unique)})
    return [pool[int(i)] for i in g.integers(0, len(pool), n)]


def test_pseudonymize_against_dict_bruteforce():
    g = np.random.default_rng(11)
    names = ["IP_ADDRESS", "HOSTNAME", "CVE_ID"]
    key = bytes(g.integers(0, 256, 32).astype(np.uint8))
    for slug_len in [0, 1, 10, 63, 64]:
        strs = _random_spans(g, 3000, 700)
        types = g.integers(0, 3, len(strs)).astype(np.uint8)
        sb, so = _csr(strs)
        c = crypto.Cache(nbuckets=257)
        r = c.pseudonymize(sb, so, types, key, slug_len, names)
        seen = {}
        pos = 0
        for i, s in enumerate(strs):
            first = s not in seen
            if first:
                seen[s] = len(seen)
            assert r["hit"][i] == (0 if first else 1)
            assert r["uid"][i] == seen[s]
            dig = pyhmac.new(key, s, hashlib.sha256)
            assert bytes(r["digests"][i]) == dig.digest()
            tok = ("[" + names[types[i]] + "_" + dig.hexdigest()[:slug_len] + "]").encode()
            assert r["out_offsets"][i] == pos
            assert bytes(r["out_tokens"][pos:pos + len(tok)]) == tok
            assert re.fullmatch(rb"\[[A-Z0-9_]+_[0-9a-f]{%d}\]" % slug_len, tok)   # PAPER.md L44 surface form
            pos += len(tok)
        assert r["out_offsets"][-1] == pos
        st = c.stats()
        assert st == {"n_unique": len(seen), "n_lookups": len(strs), "n_hits": len(strs) - len(seen)}
        # uid dense in first-occurrence order; export row = (original_name, full_hash)
        for s, u in list(seen.items())[:50]:
            b, d = c.entry(u)
            assert b == s and d == pyhmac.new(key, s, hashlib.sha256).digest()
        c.close()


def test_referential_integrity_and_split_invariance():
    g = np.random.default_rng(12)
    names = ["A", "B"]
    key1, key2 = b"\x01" * 32, b"\x02" * 32
    strs = _random_spans(g, 2000, 300, lo=1)
    types = np.zeros(len(strs), np.uint8)
    sb, so = _csr(strs)
    whole = crypto.Cache().pseudonymize(sb, so, types, key1, 10, names)
    # same call split in three: same hit/uid/pseudonyms (cache persists across calls)
    c = crypto.Cache()
    cuts = [0, 500, 1300, 2000]
    hit, uid, toks = [], [], []
    for a, b in zip(cuts[:-1], cuts[1:]):
        psb, pso = _csr(strs[a:b])
        r = c.pseudonymize(psb, pso, types[a:b], key1, 10, names)
        hit.append(r["hit"]); uid.append(r["uid"]); toks.append(bytes(r["out_tokens"]))
    assert np.array_equal(np.concatenate(hit), whole["hit"])
    assert np.array_equal(np.concatenate(uid), whole["uid"])
    assert b"".join(toks) == bytes(whole["out_tokens"])
    # second pass over the same spans: all hits, same tokens
    r2 = c.pseudonymize(sb, so, types, key1, 10, names)
    assert r2["hit"].all() and bytes(r2["out_tokens"]) == bytes(whole["out_tokens"])
    # another key on the same cache is refused; on a fresh cache every full digest differs
    with pytest.raises(KeyError):
        c.pseudonymize(sb, so, types, key2, 10, names)
    other = crypto.Cache().pseudonymize(sb, so, types, key2, 10, names)
    assert not (other["digests"] == whole["digests"]).all(axis=1).any()
    # same entity at any position -> same pseudonym
    first = {}
    for i, s in enumerate(strs):
        tok = bytes(whole["out_tokens"][whole["out_offsets"][i]:whole["out_offsets"][i + 1]])
        assert first.setdefault(s, tok) == tok


def test_empty_inputs_and_zero_length_entity():
    c = crypto.Cache()
    r = c.pseudonymize(np.zeros(0, np.uint8), np.zeros(1, np.int64), np.zeros(0, np.uint8), b"k", 10, ["T"])
    assert r["out_offsets"].tolist() == [0] and r["out_tokens"].size == 0
    sb, so = _csr([b"", b"x", b""])
    r = c.pseudonymize(sb, so, None, b"k", 4, ["T"])
    assert r["hit"].tolist() == [0, 0, 1]
    assert bytes(r["out_tokens"][:8]) == b"[T_" + pyhmac.new(b"k", b"", hashlib.sha256).hexdigest()[:4].encode() + b"]"


def test_hmac_batch_matches_single():
    strs = [b"a", b"", b"x" * 200]
    sb, so = _csr(strs)
    d = crypto.hmac_batch(b"key", sb, so)
    for i, s in enumerate(strs):
        assert bytes(d[i]) == pyhmac.new(b"key", s, hashlib.sha256).digest()
