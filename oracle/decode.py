"""TEST INFRASTRUCTURE -- BIO span decode, window stitching, span byte gather (pure Python loops).

The paper gives no decoder: PAPER.md L43 names NER detection, L133/L170 only admit
"truncation" and "span-boundary differences".  BASELINE.json north_star ¶1 asks for
"Per-token argmax and BIO span decoding"; SURVEY.md §8(c) O3 fixes the reading followed here
(S9 label map 0=O, 2t+1=B-t, 2t+2=I-t; S11 lenient starts, token level, midpoint ownership of
the 128-token window overlap; windows of 510 content tokens + [CLS]/[SEP], stride 382).

Pins: tests/test_oracle_decode.py (the ten hand-worked rows of SURVEY §8(c) O3 stored in
tests/golden/bio_cases.txt, an independent regex-style re-derivation on exhaustive label
strings, every-token-kept-exactly-once and boundary-independence of the stitch).
"""
import numpy as np

META_RECORD, META_CSTART, META_CEND, META_FLAGS = 0, 1, 2, 3
FLAG_KEEP = 1

WINDOW_CONTENT = 510   # content tokens per window (+ [CLS] and [SEP] = 512)
WINDOW_OVERLAP = 128
WINDOW_STRIDE = WINDOW_CONTENT - WINDOW_OVERLAP  # 382


def decode_spans(labels, meta):
    """O3.  labels int[T]; meta int[T,4] = (record_id, char_start, char_end, flags).

    Returns a list of (record_id, char_start, char_end, type) in order of the first token.
    """
    spans = []
    open_span = None          # [record, char_start, char_end, type]
    prev = None               # index of the previous KEPT token
    for j in range(len(labels)):
        if not (int(meta[j][META_FLAGS]) & FLAG_KEEP):
            continue          # transparent: label never read
        lab = int(labels[j])
        rec = int(meta[j][META_RECORD])
        prev_same = prev is not None and int(meta[prev][META_RECORD]) == rec
        if lab > 0:
            typ = (lab - 1) // 2
            is_i = (lab % 2) == 0
            cont = (is_i and prev_same and int(labels[prev]) > 0
                    and (int(labels[prev]) - 1) // 2 == typ)
            if cont:
                open_span[2] = int(meta[j][META_CEND])
            else:
                if open_span is not None:
                    spans.append(tuple(open_span))
                open_span = [rec, int(meta[j][META_CSTART]), int(meta[j][META_CEND]), typ]
        else:
            if open_span is not None:
                spans.append(tuple(open_span))
                open_span = None
        prev = j
    if open_span is not None:
        spans.append(tuple(open_span))
    return spans


def num_windows(n):
    """W = 1 if n <= 510 else 1 + ceil((n - 510) / 382)."""
    if n <= WINDOW_CONTENT:
        return 1
    return 1 + -(-(n - WINDOW_CONTENT) // WINDOW_STRIDE)


def window_plan(n):
    """For a record of n content tokens: list of (lo, hi, keep[lo:hi]) per window.

    Window w holds content tokens [382 w, min(382 w + 510, n)).  A token g lying in windows
    w and w+1 is kept in w iff g < 382 (w+1) + 64, else in w+1 (midpoint rule)."""
    out = []
    W = num_windows(n)
    for w in range(W):
        lo = WINDOW_STRIDE * w
        hi = min(lo + WINDOW_CONTENT, n)
        keep = []
        for g in range(lo, hi):
            k = True
            if w + 1 < W and g >= WINDOW_STRIDE * (w + 1):          # shared with the next window
                k = g < WINDOW_STRIDE * (w + 1) + WINDOW_OVERLAP // 2
            if w > 0 and g < WINDOW_STRIDE * (w - 1) + WINDOW_CONTENT:  # shared with the previous
                k = k and not (g < WINDOW_STRIDE * w + WINDOW_OVERLAP // 2)
            keep.append(k)
        out.append((lo, hi, keep))
    return out


def gather_spans(text, record_offsets, spans):
    """span_bytes[off_s : off_s+len_s] = text[rec_off[record_id] + char_start : ... + char_end]."""
    offs = [0]
    chunks = []
    for (rec, cs, ce, _t) in spans:
        base = int(record_offsets[rec])
        chunks.append(bytes(bytearray(text[base + cs: base + ce])))
        offs.append(offs[-1] + (ce - cs))
    data = np.frombuffer(b"".join(chunks), dtype=np.uint8) if chunks else np.zeros(0, np.uint8)
    return data, np.asarray(offs, np.int64)


def splice_records(text, record_offsets, spans, out_tokens, out_offsets):
    """Stage 5 of the paper's pipeline ("only sensitive values replaced", schema preserved) restricted to
    the text of a record: every record's bytes with each span [char_start, char_end) replaced by its pseudonym token
    (SURVEY.md §8(f) NEXT-1).  spans are in stream order (records ascending, char_start ascending inside a record) and
    do not overlap; out_tokens / out_offsets are the CSR of their pseudonyms.  Written as the plain definition: walk
    each record left to right, copy what lies between spans, emit the token in place of each span.

    Returns (bytes uint8[], int64[R+1] offsets of the rewritten records)."""
    R = len(record_offsets) - 1
    per_rec = [[] for _ in range(R)]
    for s, (rec, cs, ce, _t) in enumerate(spans):
        per_rec[rec].append((cs, ce, s))
    pieces, offs = [], [0]
    for r in range(R):
        base, end = int(record_offsets[r]), int(record_offsets[r + 1])
        body = bytes(bytearray(text[base:end]))
        cur, out = 0, []
        for cs, ce, s in per_rec[r]:
            if cs < cur or ce < cs or ce > len(body):
                raise ValueError("spans must be ordered, non-overlapping and inside their record")
            out.append(body[cur:cs])
            out.append(bytes(bytearray(out_tokens[int(out_offsets[s]):int(out_offsets[s + 1])])))
            cur = ce
        out.append(body[cur:])
        rec_bytes = b"".join(out)
        pieces.append(rec_bytes)
        offs.append(offs[-1] + len(rec_bytes))
    data = np.frombuffer(b"".join(pieces), dtype=np.uint8) if offs[-1] else np.zeros(0, np.uint8)
    return data, np.asarray(offs, np.int64)
