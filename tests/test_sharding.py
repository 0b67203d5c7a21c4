"""CPU-only cover of the N>1 path: record sharding, throughput reduction and the end-of-stream
mapping-table merge, on a world_size-2 `gloo` process group.  Per-rank pseudonyms come from the oracle here
(the GPU path is checked against the same oracle in tests/test_gpu_*.py)."""
import os
import socket

import numpy as np
import torch.multiprocessing as mp

from paper_2606_15650_b200 import sharding


def test_shard_range_partitions():
    for n in (0, 1, 7, 64, 70951):
        for world in (1, 2, 3, 8):
            parts = [sharding.shard_range(n, r, world) for r in range(world)]
            assert parts[0][0] == 0 and parts[-1][1] == n
            assert all(parts[i][1] == parts[i + 1][0] for i in range(world - 1))
            sizes = [b - a for a, b in parts]
            assert max(sizes) - min(sizes) <= 1


def test_shard_by_tokens_balances():
    rng = np.random.default_rng(0)
    t = np.minimum(rng.lognormal(np.log(1000), 1.1, 5000), 16384).astype(np.int64) + 8
    for world in (1, 2, 4, 8):
        cuts = sharding.shard_by_tokens(t, world)
        assert cuts[0] == 0 and cuts[-1] == t.size and (np.diff(cuts) >= 0).all()
        loads = np.array([t[cuts[r]:cuts[r + 1]].sum() for r in range(world)])
        assert loads.sum() == t.sum()
        assert loads.max() <= t.sum() / world + t.max()


def _free_port():
    s = socket.socket(); s.bind(("127.0.0.1", 0)); p = s.getsockname()[1]; s.close()
    return p


def _worker(rank, world, port, q):
    import torch.distributed as dist
    from harness import gen
    from oracle import crypto
    os.environ["MASTER_ADDR"], os.environ["MASTER_PORT"] = "127.0.0.1", str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    data, off, types, key = gen.spans_config1()
    lo, hi = sharding.shard_range(off.size - 1, rank, world)
    sub, sub_off = data[off[lo]:off[hi]], off[lo:hi + 1] - off[lo]
    oc = crypto.Cache()
    res = oc.pseudonymize(sub, sub_off, types[lo:hi], key.tobytes(), 10, gen.TYPE_NAMES_4)
    rows = [oc.entry(u) for u in range(oc.stats()["n_unique"])]
    merged = sharding.merge_mapping_tables(rows)
    units, sec = sharding.aggregate_throughput(hi - lo, 1.0 + rank)
    toks = [bytes(res["out_tokens"][res["out_offsets"][i]:res["out_offsets"][i + 1]]) for i in range(hi - lo)]
    ents = [bytes(sub[sub_off[i]:sub_off[i + 1]]) for i in range(hi - lo)]
    q.put((rank, len(merged), units, sec, dict(zip(ents, zip(toks, types[lo:hi].tolist())))))
    dist.destroy_process_group()


def test_gloo_world2_no_exchange_needed():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    got = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (_, m0, u0, s0, d0), (_, m1, u1, s1, d1) = got
    assert m0 == m1 == 700                      # 700 distinct strings in config 1, merged across ranks
    assert u0 == u1 == 1000.0 and s0 == s1 == 2.0   # sum of units, max of seconds
    # referential integrity across ranks without communication: same entity -> same slug on both ranks
    common = set(d0) & set(d1)
    assert len(common) > 20
    for e in common:
        slug0 = d0[e][0].rsplit(b"_", 1)[1]
        slug1 = d1[e][0].rsplit(b"_", 1)[1]
        assert slug0 == slug1


def test_bench_gpus_flag_launches_that_many_ranks():
    """`python bench.py --gpus 2` without torchrun re-executes itself under torch.distributed.run with two ranks (S8e); checked
    on the CPU box with the reference arm (rank 0 prints the line, rank 1 exits without work), and a --gpus / WORLD_SIZE
    mismatch fails loudly."""
    import json
    import os
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    env = {k: v for k, v in os.environ.items() if k not in ("WORLD_SIZE", "RANK", "LOCAL_RANK")}
    out = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--gpus", "2", "--impl", "reference", "--headline-only",
                          "--steps", "1", "--warmup", "0"], capture_output=True, text=True, env=env, timeout=600)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [ln for ln in out.stdout.strip().splitlines() if ln.startswith("{")]
    assert len(lines) == 1                                   # one JSON line in total, from rank 0
    d = json.loads(lines[0])
    assert d["n_gpus"] == 2 and d["impl"] == "reference" and d["value"] > 0
    bad = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--gpus", "2", "--impl", "reference", "--headline-only"],
                         capture_output=True, text=True, env=dict(env, WORLD_SIZE="3"), timeout=120)
    assert bad.returncode != 0 and "does not match WORLD_SIZE" in (bad.stderr + bad.stdout)
