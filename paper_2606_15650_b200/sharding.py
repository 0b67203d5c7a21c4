"""Host-side multi-GPU plumbing: one process per GPU, records sharded across ranks, NO
data-path collective -- sequences/records are independent (A1-A10) and a pseudonym is a pure function of
(key, entity), so referential integrity holds across GPUs without any exchange.  The only
collectives are (a) the throughput reduction bench.py reports (sum of units, max of seconds) and (b) the
optional end-of-stream all-gather of each rank's (entity, digest) rows into one mapping table (the SQLite
hand-off of PAPER.md L52).  Works on `nccl` (CUDA tensors) and `gloo` (CPU tensors; tests/test_sharding.py).
"""
import numpy as np


def shard_range(n_units, rank, world):
    """Contiguous balanced split of n_units: ranks < n_units % world get one extra.  Returns (lo, hi)."""
    if world <= 0 or not (0 <= rank < world) or n_units < 0:
        raise ValueError("bad shard arguments")
    q, r = divmod(n_units, world)
    lo = rank * q + min(rank, r)
    return lo, lo + q + (1 if rank < r else 0)


def shard_by_tokens(tokens_per_record, world):
    """Token-balanced contiguous split of a record stream: cut points at the multiples of total/world of the
    running token count (records stay whole and in stream order, so each rank's cache sees a contiguous part
    of the stream).  Returns int64[world + 1] record boundaries."""
    t = np.asarray(tokens_per_record, np.int64)
    csum = np.concatenate([[0], np.cumsum(t)])
    total = int(csum[-1])
    cuts = np.zeros(world + 1, np.int64)
    for r in range(1, world):
        cuts[r] = int(np.searchsorted(csum, total * r / world, side="left"))
    cuts[world] = t.size
    return np.maximum.accumulate(cuts)


def aggregate_throughput(units_local, seconds_local, device=None):
    """(sum over ranks of units, max over ranks of seconds).  Without an initialised process group: identity."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(units_local), float(seconds_local)
    dev = device if device is not None else ("cuda" if dist.get_backend() == "nccl" else "cpu")
    u = torch.tensor([float(units_local)], dtype=torch.float64, device=dev)
    s = torch.tensor([float(seconds_local)], dtype=torch.float64, device=dev)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    dist.all_reduce(s, op=dist.ReduceOp.MAX)
    return float(u.item()), float(s.item())


def merge_mapping_tables(local_rows):
    """End-of-stream merge of the per-rank mapping tables.  local_rows: list of (entity bytes, digest bytes).
    All-gathers the rows, deduplicates by entity in (rank, local uid) order and checks that every rank derived
    the same digest for the same entity (referential integrity across GPUs).  Returns the merged list."""
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        gathered = [None] * dist.get_world_size()
        dist.all_gather_object(gathered, list(local_rows))
    else:
        gathered = [list(local_rows)]
    merged, seen = [], {}
    for rows in gathered:
        for ent, dig in rows:
            if ent in seen:
                if seen[ent] != dig:
                    raise RuntimeError("referential integrity violated: two digests for one entity")
                continue
            seen[ent] = dig
            merged.append((ent, dig))
    return merged
