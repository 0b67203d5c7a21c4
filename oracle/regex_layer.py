"""TEST INFRASTRUCTURE -- oracle of the regex detector and of the regex / NER span merge.

PAPER.md L43 (§II stage 2): detection combines the transformer NER with "21 custom regex patterns" (IPv4/6, URL,
hostname, hashes, certificates, CVE/CPE, credentials ...); L170 notes that the standalone strategy loses recall "for
lack of overlap resolution".  The paper prints neither the patterns nor the matching rules, so this build fixes them
(readings D17-D19):

  D17  pattern set = PATTERNS below, one per synthetic entity kind of harness/gen.py (shapes only);
  D18  matching = leftmost-longest over all patterns, non-overlapping, left to right inside one record; a match must
       start and end at a word boundary (the byte before / after is not [0-9A-Za-z_]); ties between patterns of equal
       length go to the lowest pattern index;
  D19  merge = every regex span is kept; an NER span is kept iff it overlaps no regex span of its record; the result is
       ordered by (record, char_start).

Written as the plain definition: for every start position try every end position with `re.fullmatch` -- no automaton,
nothing shared with paper_2606_15650_b200/regex_dfa.py.  Pins: tests/test_oracle_regex.py (hand-worked records,
`re.finditer` with look-arounds on patterns whose greedy match is the longest one, invariants).
"""
import re

import numpy as np

# (type name, pattern) in priority order; restricted syntax (literals, classes, groups, |, ?, *, +, {m,n})
PATTERNS = [
    ("IP_ADDRESS", r"(?:[0-9]{1,3}\.){3}[0-9]{1,3}"),
    ("IPV6_ADDRESS", r"(?:[0-9a-f]{1,4}:){7}[0-9a-f]{1,4}"),
    ("HOSTNAME", r"(?:[a-z0-9]+\.)+(?:example|internal|corp|lan|test|invalid)"),
    ("CVE_ID", r"CVE-[0-9]{4}-[0-9]{4,7}"),
    ("MAC_ADDRESS", r"(?:[0-9a-f]{2}:){5}[0-9a-f]{2}"),
    ("SERIAL_NUMBER", r"[0-9a-f]{16,32}"),
]
MAX_MATCH = 80          # no pattern above matches more than this many bytes... except HOSTNAME, capped here (D18)
_WORD = frozenset(b"0123456789ABCDEFGHIJKLMNOPQRSTUVWXYZabcdefghijklmnopqrstuvwxyz_")


def scan_record(body, patterns=PATTERNS, max_match=MAX_MATCH):
    """body: bytes of one record.  Returns [(char_start, char_end, pattern_index)] by rule D18."""
    comp = [re.compile(p.encode()) for _n, p in patterns]
    out, s, n = [], 0, len(body)
    while s < n:
        best = None
        if s == 0 or body[s - 1] not in _WORD:
            for e in range(min(n, s + max_match), s, -1):              # longest end first
                if e < n and body[e] in _WORD:
                    continue
                for k, c in enumerate(comp):
                    if c.fullmatch(body, s, e):
                        best = (s, e, k)
                        break
                if best:
                    break
        if best:
            out.append(best)
            s = best[1]
        else:
            s += 1
    return out


def scan_records(text, record_offsets, patterns=PATTERNS, max_match=MAX_MATCH):
    """All records of a batch: [(record_id, char_start, char_end, pattern_index)] in stream order."""
    buf = bytes(bytearray(text))
    spans = []
    for r in range(len(record_offsets) - 1):
        a, b = int(record_offsets[r]), int(record_offsets[r + 1])
        spans += [(r, cs, ce, k) for cs, ce, k in scan_record(buf[a:b], patterns, max_match)]
    return spans


def merge_spans(ner_spans, regex_spans):
    """Rule D19.  Both lists hold (record_id, char_start, char_end, type) in stream order."""
    kept = []
    for (r, cs, ce, t) in ner_spans:
        clash = any(rr == r and cs2 < ce and cs < ce2 for (rr, cs2, ce2, _t) in regex_spans)
        if not clash:
            kept.append((r, cs, ce, t))
    return sorted(kept + list(regex_spans), key=lambda s: (s[0], s[1]))
