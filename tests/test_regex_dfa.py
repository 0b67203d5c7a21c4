"""Host logic of NEXT-4: the regex -> DFA compiler (paper_2606_15650_b200/regex_dfa.py).

The tables are walked here by a small interpreter that applies rule D18 (word boundaries, longest match, lowest pattern
index, max_match) and compared with the oracle's brute-force `re.fullmatch` scan; the interpreter lives in the test, the
product has no CPU scan."""
import struct

import numpy as np
import pytest

from oracle import regex_layer as rx
from paper_2606_15650_b200 import regex_dfa


def parse_blob(blob):
    magic, ns, nc, npat, mm, _a, _b, _c = struct.unpack_from("<8I", blob, 0)
    assert magic == regex_dfa.MAGIC
    o = 32
    class_of = np.frombuffer(blob, np.uint8, 256, o); o += 256
    is_word = np.frombuffer(blob, np.uint8, 256, o); o += 256
    types = np.frombuffer(blob, np.uint8, 256, o); o += 256
    accept = np.frombuffer(blob, "<i2", ns, o); o += (2 * ns + 3) // 4 * 4
    trans = np.frombuffer(blob, "<u2", ns * nc, o).reshape(ns, nc); o += 2 * ns * nc
    assert o == len(blob)
    return dict(class_of=class_of, is_word=is_word, types=types, accept=accept, trans=trans, max_match=mm, n_patterns=npat)


def walk(t, body):
    """[(char_start, char_end, pattern)] by rule D18 from the tables."""
    out, s, n = [], 0, len(body)
    while s < n:
        best = None
        if s == 0 or not t["is_word"][body[s - 1]]:
            st = 1
            for i in range(min(t["max_match"], n - s)):
                st = int(t["trans"][st, t["class_of"][body[s + i]]])
                if st == 0:
                    break
                e = s + i + 1
                if t["accept"][st] >= 0 and (e == n or not t["is_word"][body[e]]):
                    best = (s, e, int(t["accept"][st]))
        if best:
            out.append(best)
            s = best[1]
        else:
            s += 1
    return out


def test_default_pattern_set_matches_oracle():
    blob = regex_dfa.compile_patterns([(k, p) for k, (_n, p) in enumerate(rx.PATTERNS)], rx.MAX_MATCH)
    t = parse_blob(blob)
    assert t["n_patterns"] == len(rx.PATTERNS) and t["trans"].shape[0] < 2000
    assert not t["trans"][0].any() and t["accept"][0] < 0 and t["accept"][1] < 0
    rng = np.random.default_rng(17)
    alphabet = np.frombuffer(b"0123456789abcdefCVE-.: xlanitrpoms_", np.uint8)
    plants = [b"10.20.30.40", b"CVE-1999-0001", b"aa:bb:cc:dd:ee:ff", b"0123456789abcdef0123", b"1:2:3:4:5:6:7:8",
              b"db1.core.internal", b"x.lan", b"a.b.c.example", b"fe80:0:0:0:1:2:3:4", b"999.999.999.999.test"]
    for trial in range(60):
        body = bytes(rng.choice(alphabet, 400).astype(np.uint8))
        for k in range(4):
            pos = int(rng.integers(0, 340))
            pl = plants[int(rng.integers(0, len(plants)))]
            sep = b" " if rng.random() < 0.7 else b""
            body = body[:pos] + sep + pl + sep + body[pos + len(pl) + 2 * len(sep):]
        assert walk(t, body) == rx.scan_record(body), body
    # a hostname longer than max_match is cut out by the cap exactly as in the oracle
    long_host = b"a" * 100 + b".lan and " + b"b" * 70 + b".lan"
    assert walk(t, long_host) == rx.scan_record(long_host) and len(walk(t, long_host)) == 1


@pytest.mark.parametrize("pats", [
    [r"ab|abc|abcd", r"[a-c]+d?"],
    [r"(?:x|yz){2,3}", r"x{3,}", r"\d+\.\d*"],
    [r"[^ \t]{3}", r"\w+@\w+(?:\.\w+)+"],
    [r"a?b?c?d", r"(?:ab)*c", r"\x41\x42"],
    [r"[a\-z]+", r"[]x]+", r"a.c"],
])
def test_syntax_coverage_against_oracle(pats):
    named = [("P%d" % k, p) for k, p in enumerate(pats)]
    t = parse_blob(regex_dfa.compile_patterns([(k, p) for k, p in enumerate(pats)], 40))
    rng = np.random.default_rng(len(pats[0]))
    alphabet = np.frombuffer(b"abcdxyz019.@ -]AB\n", np.uint8)
    for trial in range(40):
        body = bytes(rng.choice(alphabet, 120).astype(np.uint8))
        assert walk(t, body) == rx.scan_record(body, named, 40), (pats, body)


def test_rejects_what_it_cannot_compile():
    for bad in [r"^abc", r"abc$", r"a*?", r"(?=x)y", r"(a)\1", r"\bword", r"[z-a]", r"a{3,2}", r"(ab", r"ab)", r"*a", r"x*"]:
        with pytest.raises(ValueError):
            regex_dfa.compile_patterns([(0, bad)])
    with pytest.raises(ValueError):
        regex_dfa.compile_patterns([])
    with pytest.raises(ValueError):
        regex_dfa.compile_patterns([(0, "a")], max_match=300)


def test_minimisation_merges_equivalent_states():
    # (a|b)c and [ab]c are the same language: identical tables; 4 states = dead, start, after [ab], accept
    c1, a1, t1 = regex_dfa.compile_tables([r"(?:a|b)c"])
    c2, a2, t2 = regex_dfa.compile_tables([r"[ab]c"])
    assert t1.shape[0] == 4 and np.array_equal(a1, a2) and np.array_equal(t1[:, c1[list(b"abc ")]], t2[:, c2[list(b"abc ")]])


def _random_pattern(rng, depth=0):
    """A random pattern of the restricted grammar.  Unbounded repeats are put on single atoms only: the ORACLE is a
    backtracking `re.fullmatch` per (start, end) pair, and nested or ambiguous stars make it exponential -- the compiler has no
    such problem, but the test has to finish."""
    atoms = ["a", "b", "c", "0", "1", r"\.", "-", "[ab]", "[0-9]", "[^a ]", r"\d", "[a-c0]", "."]
    r = rng.random()
    if depth >= 3 or r < 0.35:
        node = atoms[int(rng.integers(0, len(atoms)))]
        q = rng.random()
        if q < 0.15:
            node += "+"
        elif q < 0.25:
            node += "*"
        elif q < 0.32:
            node += "{2,}"
        return node
    if r < 0.6:
        node = "".join(_random_pattern(rng, depth + 1) for _ in range(int(rng.integers(2, 4))))
    elif r < 0.85:
        node = "(?:" + "|".join(_random_pattern(rng, depth + 1) for _ in range(int(rng.integers(2, 4)))) + ")"
    else:
        node = "(?:" + _random_pattern(rng, depth + 1) + ")"
    q = rng.random()
    if q < 0.15:
        node = "(?:" + node + ")?"
    elif q < 0.3:
        lo = int(rng.integers(0, 3))
        node = "(?:" + node + "){%d,%d}" % (lo, lo + int(rng.integers(0, 2)))
    return node


def test_random_patterns_against_oracle():
    """Fuzz: random pattern sets from the restricted grammar, random bodies; the table walk must equal the oracle's
    brute-force `re.fullmatch` scan (rule D18) for every set the compiler accepts."""
    import re
    rng = np.random.default_rng(2026)
    alphabet = np.frombuffer(b"abc01.- x", np.uint8)
    done = 0
    for trial in range(400):
        pats = [_random_pattern(rng) for _ in range(int(rng.integers(1, 4)))]
        if any(re.fullmatch(p, "") for p in pats):
            with pytest.raises(ValueError):
                regex_dfa.compile_patterns(list(enumerate(pats)), 24)
            continue
        t = parse_blob(regex_dfa.compile_patterns(list(enumerate(pats)), 24))
        named = [("P%d" % k, p) for k, p in enumerate(pats)]
        for _ in range(6):
            body = bytes(rng.choice(alphabet, 60).astype(np.uint8))
            assert walk(t, body) == rx.scan_record(body, named, 24), (pats, body)
        done += 1
    assert done > 150
