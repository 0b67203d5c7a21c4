"""Host glue for streaming a record stream through the hot path in token-budgeted batches (BASELINE.json
configs[2]: 70,951 records, ~175 M window-tokens do not fit in one pass).

Outside the hot path (plain host code, like the tokenizer): it only cuts the already tokenised / windowed stream
into batches of WHOLE records -- a span may cross a window boundary but never a record boundary (reading D8), so
cutting between records changes no output -- and rebases record ids / text offsets so that each batch is a
self-contained input of anon_pipeline_host.  The entity cache persists across batches, which is what gives the
stream its hit rate ("LRU cache to amortise repeated lookups across records", L111).
"""
import numpy as np


def plan_batches(win_rec, cu_seqlens, token_budget):
    """win_rec int[B]: record of every window (non-decreasing); cu_seqlens int[B+1].  Returns a list of
    (w0, w1) window ranges, each covering whole records and at most token_budget tokens (a single record larger
    than the budget gets a batch of its own)."""
    win_rec = np.asarray(win_rec)
    cu = np.asarray(cu_seqlens, np.int64)
    B = win_rec.size
    if B == 0:
        return []
    if (np.diff(win_rec) < 0).any():
        raise ValueError("windows of one record must be adjacent and records in order")
    # first window of every record
    starts = np.flatnonzero(np.concatenate([[True], win_rec[1:] != win_rec[:-1]]))
    bounds = np.concatenate([starts, [B]])
    out, w0 = [], 0
    for k in range(1, bounds.size):
        w_next = int(bounds[k])
        if cu[w_next] - cu[w0] > token_budget and int(bounds[k - 1]) > w0:
            out.append((w0, int(bounds[k - 1])))
            w0 = int(bounds[k - 1])
    out.append((w0, B))
    return out


def slice_batch(rec, win, w0, w1):
    """Self-contained inputs of windows [w0, w1): record ids rebased to the batch, text limited to its records."""
    cu = win["cu_seqlens"]
    t0, t1 = int(cu[w0]), int(cu[w1])
    r0, r1 = int(win["win_rec"][w0]), int(win["win_rec"][w1 - 1]) + 1
    meta = np.array(win["meta"][t0:t1], np.int32, copy=True)
    meta[:, 0] -= r0
    ro = rec["rec_off"]
    return dict(token_ids=np.ascontiguousarray(win["token_ids"][t0:t1], np.int32),
                cu_seqlens=(cu[w0:w1 + 1] - cu[w0]).astype(np.int32),
                meta=meta,
                text=np.ascontiguousarray(rec["text"][int(ro[r0]):int(ro[r1])]),
                rec_off=(ro[r0:r1 + 1] - ro[r0]).astype(np.int64),
                r0=r0, r1=r1, t0=t0, t1=t1)
