"""Pins of oracle/regex_layer.py (readings D17-D19 in DESIGN.md)."""
import re

import numpy as np

from oracle import regex_layer as rx


def test_hand_worked_records():
    names = [n for n, _p in rx.PATTERNS]
    body = b"scan of 10.0.0.1 (srv1.db2.corp) found CVE-2024-12345 on 00:1a:2b:3c:4d:5e, serial 0123456789abcdef01, x10.0.0.2"
    got = [(body[s:e].decode(), names[k]) for s, e, k in rx.scan_record(body)]
    assert got == [("10.0.0.1", "IP_ADDRESS"), ("srv1.db2.corp", "HOSTNAME"), ("CVE-2024-12345", "CVE_ID"),
                   ("00:1a:2b:3c:4d:5e", "MAC_ADDRESS"), ("0123456789abcdef01", "SERIAL_NUMBER")]
    # "x10.0.0.2" does not start at a word boundary; "10.0.0.2" inside it starts after a word character: no match
    # leftmost-longest: an IPv6 address is not cut into a MAC-shaped prefix; ties go to the lower pattern index
    body = b"2001:0db8:00aa:00bb:00cc:00dd:00ee:00ff 1.2.3.4.5 CVE-2024-123"
    got = [(body[s:e].decode(), names[k]) for s, e, k in rx.scan_record(body)]
    assert got == [("2001:0db8:00aa:00bb:00cc:00dd:00ee:00ff", "IPV6_ADDRESS"), ("1.2.3.4", "IP_ADDRESS")]
    assert rx.scan_record(b"") == [] and rx.scan_record(b"no entity here, not.a.host.name") == []


def test_single_patterns_against_re_finditer():
    """For these patterns the greedy match is the longest one, so leftmost-longest with word boundaries equals
    re.finditer with look-arounds -- an independent library routine."""
    rng = np.random.default_rng(3)
    alphabet = b"0123456789abcdefCVE-.: x"
    for name, pat in rx.PATTERNS:
        if name == "HOSTNAME":
            continue
        lib = re.compile(rb"(?<![0-9A-Za-z_])(?:" + pat.encode() + rb")(?![0-9A-Za-z_])")
        for trial in range(30):
            body = bytes(rng.choice(np.frombuffer(alphabet, np.uint8), 300).astype(np.uint8))
            # plant a few well-formed entities
            plants = [b"10.20.30.40", b"CVE-1999-0001", b"aa:bb:cc:dd:ee:ff", b"0123456789abcdef0123", b"1:2:3:4:5:6:7:8"]
            for k in range(3):
                pos = int(rng.integers(0, 250))
                pl = plants[int(rng.integers(0, len(plants)))]
                body = body[:pos] + b" " + pl + b" " + body[pos + len(pl) + 2:]
            want = [(m.start(), m.end()) for m in lib.finditer(body)]
            got = [(s, e) for s, e, _k in rx.scan_record(body, [(name, pat)])]
            assert got == want, (name, body)


def test_invariants_and_records():
    rng = np.random.default_rng(5)
    recs = []
    for r in range(12):
        words = []
        for k in range(int(rng.integers(0, 30))):
            c = int(rng.integers(0, 6))
            words.append([b"alpha", b"192.168.%d.%d" % (k, r), b"CVE-2020-%04d" % (k * 7), b"de:ad:be:ef:%02x:%02x" % (k, r),
                          b"node%d.lab.internal" % k, b"%032x" % (k * 7919 + r)][c])
        recs.append(b" ".join(words))
    text = np.frombuffer(b"".join(recs), np.uint8)
    off = np.array([0] + list(np.cumsum([len(b) for b in recs])), np.int64)
    spans = rx.scan_records(text, off)
    assert len(spans) > 50
    last = {}
    for (r, cs, ce, k) in spans:
        body = recs[r]
        assert 0 <= cs < ce <= len(body) and ce - cs <= rx.MAX_MATCH
        assert re.fullmatch(rx.PATTERNS[k][1].encode(), body[cs:ce])
        assert cs == 0 or body[cs - 1:cs] not in [bytes([c]) for c in rx._WORD]
        assert cs >= last.get(r, 0)                                   # ordered, non-overlapping inside a record
        last[r] = ce
    # a record boundary is a hard boundary: scanning the concatenation record by record == scanning each alone
    assert spans == [(r, cs, ce, k) for r in range(len(recs)) for cs, ce, k in rx.scan_record(recs[r])]


def test_merge_rule():
    ner = [(0, 0, 4, 1), (0, 10, 20, 2), (0, 30, 35, 0), (1, 5, 9, 3), (2, 0, 3, 1)]
    rgx = [(0, 15, 25, 4), (0, 35, 40, 5), (1, 0, 5, 0), (1, 8, 12, 0)]
    got = rx.merge_spans(ner, rgx)
    # (0,10,20) overlaps (0,15,25): dropped; (0,30,35) only touches (0,35,40): kept; (1,5,9) overlaps (1,8,12): dropped
    assert got == [(0, 0, 4, 1), (0, 15, 25, 4), (0, 30, 35, 0), (0, 35, 40, 5), (1, 0, 5, 0), (1, 8, 12, 0), (2, 0, 3, 1)]
    assert rx.merge_spans([], rgx) == rgx and rx.merge_spans(ner, []) == ner
