#!/usr/bin/env python
"""bench.py -- throughput of the AnonShield hot path (A1-A13) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload base|large|stream|pseudonym|fields|modern]
                    [--headline-only] [--impl reference]

A "step" is one pass of the whole hot path over one batch of seeded synthetic input: anon_ner_forward ->
anon_decode_spans -> anon_gather_spans -> anon_pseudonymize (cache cleared first, so every step inserts and
HMACs the same entities).  The timed workload of the ONE JSON line is BASELINE.json configs[1] (BERT-base shape, BF16,
4,096 packed sequences, lognormal lengths): `value` = tokens/s with inputs resident in HBM; `e2e` = the same metric through
anon_pipeline_host with pinned HOST buffers (H2D + D2H inside the timed region).

At N = 1 with the default workload the same process then also measures, each in its own timed region, and embeds as extra
keys of the same line (skipped with --headline-only or when the time budget --extra-budget-s runs out):
  "stream"    BASELINE.json configs[2]: the full 70,951-record stream (records/s, seconds, e2e text in -> text out)
  "pseudonym" configs[4]: 50 M spans through the hash cache + HMAC-SHA256 + write-back (spans/s, e2e with host span buffers,
              the C oracle on the full 50 M spans as cpu_baseline)
  "large"     configs[3]: 24 x 1024 encoder, vocab 250,002 (tokens/s)
  "fields"    S8f NEXT-2: field spans -> gather -> pseudonymize -> splice over the stream's text, no encoder (KB/s, spans/s)
Each carries its own `roofline` (and `cpu_baseline` / `e2e` where the metric has one).  `--workload X` runs one of them alone
as the main line.  Under torchrun (N > 1) every rank runs its own shard of the same size (weak scaling, no data-path
collective); time = max over ranks, value = sum of tokens / that time.  `--gpus N` without torchrun re-executes itself under
`python -m torch.distributed.run --nproc-per-node N`.
"""
import argparse
import hashlib
import json
import os
import socket
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from harness import gen  # noqa: E402  (seeded input generators: no arithmetic of the method)

KEY = bytes((7 * i + 3) & 255 for i in range(32))
SLUG_LEN = 10
PLANTED = gen.PLANTED_DEEP       # W2 planted-detector weights (DESIGN.md input recipe): survives 12 and 24 layers
T_START = time.time()


def log(*a):
    print(*a, file=sys.stderr, flush=True)


# ---- clocks ------------------------------------------------------------------------------------------------
class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms DURING the timed region (B200_PROFILING.md)."""
    FIELDS = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
              "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
              "clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_id):
        self.lines, self.proc = [], None
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(gpu_id), "--query-gpu=" + self.FIELDS,
                                          "--format=csv,noheader,nounits", "-lms", "200"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._pump, daemon=True)
            self.th.start()
        except OSError:
            self.proc = None

    def _pump(self):
        for ln in self.proc.stdout:
            self.lines.append(ln.strip())

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, smax, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.lines:
            p = [x.strip() for x in ln.split(",")]
            if len(p) < 7:
                continue
            try:
                sm.append(float(p[0])); smax.append(float(p[1])); pw.append(float(p[2]))
            except ValueError:
                continue
            for n, v in zip(names, p[3:7]):
                if v == "Active":
                    reasons.add(n)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(smax) if smax else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            d = json.load(f)
        return {"hbm_gbs": d["hbm_gbs"], "bf16_tflops": d["bf16_tflops"],
                "bf16_tflops_sustained": d.get("bf16_tflops_sustained", d["bf16_tflops"]), "source": "measured"}
    return {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0, "source": "fallback"}



GEMM_CLASSES = {"gemm_qkv": "QKV projection, +bias (N = 3H, K = H)", "gemm_out": "out-projection, +bias +FP32 residual (N = K = H)",
                "gemm_ffn1": "FFN up, +bias +erf-GELU (N = F, K = H)", "gemm_ffn2": "FFN down, +bias +FP32 residual (N = H, K = F)"}
def ncu_traffic_base():
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of the four GEMMs at the DEFAULT workload, from the `ncu --set
    full` capture recorded in profiles/traffic_base.json.txt.  The file names the commit and the SHA-256 of the kernel source it
    was taken from; if csrc/gemm_tcgen05.cu has changed since, the numbers are stale and `traffic` is null."""
    try:
        with open(os.path.join(ROOT, "profiles", "traffic_base.json.txt")) as f:
            rec = json.load(f)
        with open(os.path.join(ROOT, "paper_2606_15650_b200", "csrc", "gemm_tcgen05.cu"), "rb") as f:
            sha = hashlib.sha256(f.read()).hexdigest()
        return rec["traffic_bytes_per_launch"] if rec.get("gemm_tcgen05_cu_sha256") == sha else None
    except (OSError, ValueError, KeyError):
        return None


def gemm_rooflines(prof, peaks, traffic=None):
    """Per-GEMM achieved TFLOP/s from the context's event timing, the class total, and the `roofline` object of the
    dominant one (largest share of the timed region)."""
    peak = peaks["bf16_tflops_sustained"]
    per, tot_ms, tot_fl, tot_n = {}, 0.0, 0.0, 0
    for k in GEMM_CLASSES:
        ms, fl, n = prof[k]
        tot_ms += ms; tot_fl += fl; tot_n += n
        if ms > 0:
            per[k] = {"ms": ms, "launches": n, "tflops": fl / (ms * 1e-3) / 1e12, "frac": fl / (ms * 1e-3) / 1e12 / peak}
    top = max(per, key=lambda k: per[k]["ms"])
    ms, fl, n = prof[top]
    achieved = fl / (ms * 1e-3) / 1e12
    roof = {"bound": "tensor", "kernel": "gemm_bf16_tcgen05_kernel: " + GEMM_CLASSES[top], "achieved": achieved, "peak": peak,
            "unit": "TFLOP/s", "frac": achieved / peak,
            "peak_source": "MEASURED_PEAKS.json bf16_tflops_sustained (%s)" % peaks["source"],
            "frac_of_burst_peak": achieved / peaks["bf16_tflops"], "frac_of_nominal_2250": achieved / 2250.0,
            "launches": n, "avg_launch_ms": ms / max(n, 1), "flops_per_launch": fl / max(n, 1),
            "traffic": (traffic or {}).get(top),
            "all_gemms": {"ms": tot_ms, "launches": tot_n, "tflops": tot_fl / (tot_ms * 1e-3) / 1e12 if tot_ms > 0 else 0.0,
                          "frac": tot_fl / (tot_ms * 1e-3) / 1e12 / peak if tot_ms > 0 else 0.0, "per_kernel": per}}
    return roof, tot_ms


# ---- workloads ---------------------------------------------------------------------------------------------
def encoder_workload(name, rank, n_records=None):
    """Seeded synthetic record stream + windows for BASELINE.json configs[1] ("base") or configs[3] ("large");
    rank r draws its own shard with seed + 1000 r (weak scaling)."""
    if name == "base":
        desc = gen.DESCS["base"]
        rec, win = gen.workload_base(n_records=n_records or 4096, seed=gen.SEED_BASE + 2 + 1000 * rank)
        wseed = gen.SEED_BASE + 2
        label = "BASELINE.json configs[1]: BERT-base shape BF16, %d packed sequences, lognormal(median 200, cap 512)"
    elif name == "modern":       # NEXT-3: the configs[1] input recipe through the ModernBERT-base-shaped encoder (reading D20)
        desc = gen.DESCS["base_modern"]
        rec, win = gen.workload_base(n_records=n_records or 4096, seed=gen.SEED_BASE + 2 + 1000 * rank, desc=desc)
        wseed = gen.SEED_BASE + 7
        label = ("S8f NEXT-3: ModernBERT-base shape BF16 (22 layers, hidden 768, GeGLU 1152, RoPE, local window 128 in 2 of 3 "
                 "layers), %d packed sequences, lognormal(median 200, cap 512)")
    else:
        desc = gen.DESCS["large"]
        rec, win = gen.workload_large(n_seqs=n_records or 16384, seed=gen.SEED_BASE + 4 + 1000 * rank)
        wseed = gen.SEED_BASE + 4
        label = "BASELINE.json configs[3]: 24x1024 encoder BF16, vocab 250002, %d packed sequences U[32,512]"
    return desc, rec, win, wseed, label % (len(win["cu_seqlens"]) - 1)


def make_weights_for(desc, seed):
    if desc.get("arch") == 1:       # the arch-1 generator plants the shallow detector only: (alpha, beta, gamma)
        return gen.make_weights_modern(desc, seed, planted=tuple(PLANTED[:3]))
    return gen.make_weights(desc, seed, planted=PLANTED)


def pack_for(desc, w):
    return gen.pack_blob_modern(w) if desc.get("arch") == 1 else gen.pack_blob(w)


def oracle_sample_pass(w, desc, rec, win, n_seqs, names):
    """The oracle, as it stands, over the first n_seqs sequences of the workload: encoder + argmax + BIO decode +
    gather + dedup/HMAC/write-back.  Returns (tokens, spans, seconds)."""
    from oracle import crypto, decode, encoder, encoder_modern
    cu = win["cu_seqlens"]
    T = int(cu[n_seqs])
    ids, meta = win["token_ids"][:T], win["meta"][:T]
    t0 = time.perf_counter()
    logits = (encoder_modern if desc.get("arch") == 1 else encoder).forward_packed(w, desc, ids, cu[:n_seqs + 1])
    labels = encoder.argmax_labels(logits)
    spans = decode.decode_spans(labels, meta)
    sb, so = decode.gather_spans(rec["text"], rec["rec_off"], spans)
    oc = crypto.Cache()
    oc.pseudonymize(sb, so, np.asarray([s[3] for s in spans], np.uint8), KEY, SLUG_LEN, names)
    dt = time.perf_counter() - t0
    oc.close()
    return T, len(spans), dt


def blas_threads():
    try:
        from threadpoolctl import threadpool_info
        n = [i.get("num_threads", 1) for i in threadpool_info() if i.get("user_api") == "blas"]
        return max(n) if n else 1
    except Exception:
        return os.cpu_count() or 1


def seqs_for_tokens(cu, budget):
    n = int(np.searchsorted(cu, budget, side="right")) - 1
    return max(1, min(n, len(cu) - 1))


# ---- reference arm: the oracle on the host cores --------------------------------------------------------------
def reference_line(args, workload, steps, warmup):
    """The oracle, as it stands, on the host cores over a bounded sample of `workload`; returns the JSON object."""
    if workload == "pseudonym":
        return reference_pseudonym(args, steps, warmup)
    if workload == "fields":
        return reference_fields(args, steps, warmup)
    if workload == "stream":
        desc, wseed = gen.DESCS["base"], gen.SEED_BASE + 2
        rec = gen.workload_stream(n_records=64, seed=gen.SEED_BASE + 3, n_pool=300000)
        win = gen.window_records(rec)
        label = "BASELINE.json configs[2]: synthetic record stream, 510+2-token windows (first 64 records generated)"
    else:
        desc, rec, win, wseed, label = encoder_workload(workload, 0, n_records=64)
    w = make_weights_for(desc, wseed)
    names = gen.TYPE_NAMES_6
    n = seqs_for_tokens(win["cu_seqlens"], 250 if workload == "large" else 600)
    tot_t = tot_s = 0
    times = []
    for i in range(warmup + steps):
        T, S, dt = oracle_sample_pass(w, desc, rec, win, n, names)
        if i >= warmup:
            tot_t += T; tot_s += S; times.append(dt)
    sec = sum(times)
    v = tot_t / sec
    sample = "first %d sequences (%d tokens) of the workload per step" % (n, int(win["cu_seqlens"][n]))
    metric, unit = "ner_tokens_per_s", "tokens/s"
    if workload == "stream":     # records/s = tokens/s over the stream's window-tokens per record
        v = v * (len(rec["rec_off"]) - 1) / float(win["cu_seqlens"][-1])
        metric, unit = "records_per_s", "records/s"
        sample += "; tokens/s scaled by the sample's window-tokens per record"
    return {"impl": "reference", "metric": metric, "value": v, "unit": unit, "n_gpus": args.gpus,
            "steps": steps, "warmup": warmup, "ms_per_step": 1e3 * sec / steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": label, "sample": sample},
            "cpu_baseline": {"value": v, "unit": unit, "cores": blas_threads(), "kind": "oracle", "sample": sample},
            "e2e": {"value": v, "unit": unit, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "spans_per_s": tot_s / sec}


def reference_pseudonym(args, steps, warmup):
    from oracle import crypto
    n_draws = 2_000_000
    data, off, types, key, _ = gen.spans_zipf(200_000, n_draws, 7, 128, 6, gen.SEED_BASE + 5)
    times = []
    for i in range(warmup + steps):
        oc = crypto.Cache(1 << 20)
        t0 = time.perf_counter()
        oc.pseudonymize(data, off, types, key.tobytes(), SLUG_LEN, gen.TYPE_NAMES_6)
        dt = time.perf_counter() - t0
        oc.close()
        if i >= warmup:
            times.append(dt)
    sec = sum(times)
    v = n_draws * steps / sec
    sample = "2,000,000 spans Zipf(1.1) over 200,000 strings (1/25 of configs[4]) per step"
    return {"impl": "reference", "metric": "pseudonym_spans_per_s", "value": v, "unit": "spans/s", "n_gpus": args.gpus,
            "steps": steps, "warmup": warmup, "ms_per_step": 1e3 * sec / steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "u32", "data": "synthetic",
            "config": {"workload": "BASELINE.json configs[4] pseudonym-stage stress", "sample": sample},
            "cpu_baseline": {"value": v, "unit": "spans/s", "cores": 1, "kind": "oracle", "sample": sample},
            "e2e": {"value": v, "unit": "spans/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}


def reference_fields(args, steps, warmup):
    rec = gen.workload_stream(n_records=1500, seed=gen.SEED_BASE + 3, n_pool=300000)
    times, nb, ns = [], 0, 0
    for i in range(warmup + steps):
        nb, ns, dt = oracle_fields_pass(rec, 1500)
        if i >= warmup:
            times.append(dt)
    sec = sum(times)
    v = nb / 1024.0 * steps / sec
    sample = "first 1500 records of the configs[2] stream (%.1f MiB, %d field spans) per step" % (nb / 2**20, ns)
    return {"impl": "reference", "metric": "field_path_kb_per_s", "value": v, "unit": "KB/s", "n_gpus": args.gpus,
            "steps": steps, "warmup": warmup, "ms_per_step": 1e3 * sec / steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "u32", "data": "synthetic",
            "config": {"workload": "S8f NEXT-2 field path on the configs[2] records", "sample": sample},
            "cpu_baseline": {"value": v, "unit": "KB/s", "cores": 1, "kind": "oracle", "sample": sample},
            "e2e": {"value": v, "unit": "KB/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "spans_per_s": ns * steps / sec}


def run_reference(args):
    """--impl reference: rank 0 alone; the main line on args.workload, and (default workload, not --headline-only) the
    same extra keys as our arm, each on its own bounded sample with one timed step."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    out = reference_line(args, args.workload, args.steps, args.warmup)
    if args.workload == "base" and not args.headline_only:
        for name in ("stream", "pseudonym", "large", "fields"):
            t0 = time.time()
            out[name] = reference_line(args, name, 1, 0)
            log(f"[reference] {name}: {time.time() - t0:.0f}s")
    print(json.dumps(out), flush=True)


# ---- our arm ---------------------------------------------------------------------------------------------------
def dist_setup(args):
    import torch
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the hot path has no CPU fallback (use --impl reference for the oracle)")
    torch.cuda.set_device(local)
    if world > 1:
        import torch.distributed as dist
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    return world, rank, local


def barrier(world):
    import torch
    if world > 1:
        import torch.distributed as dist
        dist.barrier()
    torch.cuda.synchronize()


def gpu_id_for_smi(local):
    import torch
    try:
        u = str(torch.cuda.get_device_properties(local).uuid)
        return u if u.startswith("GPU-") else "GPU-" + u
    except Exception:
        vis = os.environ.get("CUDA_VISIBLE_DEVICES")
        return vis.split(",")[local] if vis else local


def run_encoder(args, workload=None, steps=None, warmup=None, e2e_steps=5, records=None):
    """One encoder workload (configs[1] "base", configs[3] "large", NEXT-3 "modern"); returns the JSON object (rank 0) or None."""
    import torch
    import paper_2606_15650_b200 as P
    from paper_2606_15650_b200 import sharding
    workload = workload or args.workload
    steps = steps or args.steps
    warmup = args.warmup if warmup is None else warmup
    world, rank, local = dist_setup(args)
    dev = torch.device("cuda", local)
    peaks = measured_peaks()
    t_setup = time.time()
    desc, rec, win, wseed, label = encoder_workload(workload, rank, records)
    names = gen.TYPE_NAMES_6
    w = make_weights_for(desc, wseed)
    ids, cu, meta = win["token_ids"], win["cu_seqlens"], np.ascontiguousarray(win["meta"])
    text, rec_off = rec["text"], rec["rec_off"]
    T, B, R = int(ids.size), int(cu.size - 1), int(rec_off.size - 1)
    cap = T // 2 + 1024
    out_cap = cap * 32
    ws = P.anon_workspace_bytes(desc, T, B) + 96 * T + 2 * text.size + out_cap + 40 * cap + (128 << 20)
    ctx = P.Context(local, workspace_bytes=ws)
    W = P.Weights(ctx, desc, pack_for(desc, w))
    cache = P.Cache(ctx, 1 << 20, 64 << 20)
    log(f"[rank {rank}] setup {time.time() - t_setup:.1f}s: T={T} B={B} R={R} text={text.size} ws={ws / 2**30:.1f} GiB")

    d = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(dev)
    d_ids, d_cu, d_meta, d_text, d_rec_off = d(ids), d(cu), d(meta), d(text), d(rec_off)
    labels = torch.zeros(T, dtype=torch.int32, device=dev)
    spans = torch.zeros((cap, 4), dtype=torch.int32, device=dev)
    nsp = torch.zeros(1, dtype=torch.int32, device=dev)
    span_bytes = torch.zeros(text.size + 16, dtype=torch.uint8, device=dev)
    span_off = torch.zeros(cap + 1, dtype=torch.int64, device=dev)
    span_type = torch.zeros(cap, dtype=torch.uint8, device=dev)
    out_tokens = torch.zeros(out_cap, dtype=torch.uint8, device=dev)
    out_off = torch.zeros(cap + 1, dtype=torch.int64, device=dev)
    hit = torch.zeros(cap, dtype=torch.uint8, device=dev)
    nsp_host = torch.zeros(1, dtype=torch.int32).pin_memory()
    state = {"S": 0}

    def step():
        cache.clear()
        P.anon_ner_forward(ctx, W, d_ids, d_cu, None, labels)
        P.anon_decode_spans(ctx, labels, d_meta, desc["num_labels"], spans, nsp)
        nsp_host.copy_(nsp, non_blocking=True)
        rc = ctx.sync()
        if rc:
            raise RuntimeError(f"device status {rc}")
        S = int(nsp_host[0])
        P.anon_gather_spans(ctx, d_text, d_rec_off, spans, S, span_bytes, span_off, span_type)
        P.anon_pseudonymize(ctx, cache, span_bytes, span_off[:S + 1], span_type, KEY, SLUG_LEN, names, out_tokens,
                            out_off[:S + 1], hit)
        state["S"] = S

    for _ in range(warmup):
        step()
    assert ctx.sync() == 0
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier(world)
    sampler = ClockSampler(gpu_id_for_smi(local)) if rank == 0 else None
    ctx.profile(True)
    ev0.record()
    for _ in range(steps):
        step()
    ev1.record()
    barrier(world)
    prof, launches = ctx.profile_read()
    ctx.profile(False)
    clocks = sampler.stop() if sampler else None
    sec_local = ev0.elapsed_time(ev1) / 1e3
    S = state["S"]
    tokens_all, sec = sharding.aggregate_throughput(T * steps, sec_local, dev)
    spans_all, _ = sharding.aggregate_throughput(S * steps, sec_local, dev)
    recs_all, _ = sharding.aggregate_throughput(R * steps, sec_local, dev)

    # ---- e2e: the same pass through anon_pipeline_host with pinned HOST buffers ----
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory().numpy()
    h_ids, h_cu, h_meta, h_text, h_rec_off = pin(ids), pin(cu), pin(meta), pin(text), pin(rec_off)
    bufs = dict(spans=torch.zeros((cap, 4), dtype=torch.int32).pin_memory().numpy(),
                out=torch.zeros(out_cap, dtype=torch.uint8).pin_memory().numpy(),
                off=torch.zeros(cap + 1, dtype=torch.int64).pin_memory().numpy(),
                hit=torch.zeros(cap, dtype=torch.uint8).pin_memory().numpy())

    def step_host():
        cache.clear()
        return P.anon_pipeline_host(ctx, W, cache, h_ids, h_cu, h_meta, h_text, h_rec_off, KEY, SLUG_LEN, names, cap,
                                    out_cap, want_hit=True, bufs=bufs)
    for _ in range(min(warmup, 2, e2e_steps)):
        res = step_host()
    barrier(world)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    n_e2e = max(1, min(steps, e2e_steps))
    e0.record()
    for _ in range(n_e2e):
        res = step_host()
    e1.record()
    barrier(world)
    e2e_tokens, e2e_sec = sharding.aggregate_throughput(T * n_e2e, e0.elapsed_time(e1) / 1e3, dev)
    h2d = ids.nbytes + cu.nbytes + meta.nbytes + text.nbytes + rec_off.nbytes
    Sh = len(res["spans"])
    d2h = Sh * 16 + int(res["out_tokens"].size) + (Sh + 1) * 8 + Sh + 8

    cache.close(); W.close(); ctx.close()
    del d_ids, d_cu, d_meta, d_text, d_rec_off, labels, spans, span_bytes, span_off, span_type, out_tokens, out_off, hit, bufs
    torch.cuda.empty_cache()
    if rank != 0:
        return None
    default_shape = workload == "base" and records is None
    roof, g_ms = gemm_rooflines(prof, peaks, ncu_traffic_base() if default_shape else None)
    a_ms, a_fl, a_n = prof["attention"]
    r_ms, r_by, r_n = prof["row"]
    out = {
        "metric": "ner_tokens_per_s", "value": tokens_all / sec, "unit": "tokens/s", "n_gpus": world,
        "steps": steps, "warmup": warmup, "ms_per_step": 1e3 * sec / steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "bf16", "data": "synthetic",
        "config": {"workload": label, "tokens_per_step_per_gpu": T, "records_per_step_per_gpu": R,
                   "spans_per_step_per_gpu": S,
                   "weights": "W2 planted-detector (%s), seeded random-init" % ("embedding / head triple" if desc.get("arch") == 1 else "deep variant"),
                   "l2": "inputs larger than L2 (activations %.1f GB per step stream through HBM)" % (T * 19968 / 1e9),
                   "slug_len": SLUG_LEN},
        "records_per_s": recs_all / sec, "spans_per_s": spans_all / sec,
        "clocks": clocks, "gpu_launches": launches,
        "e2e": {"value": e2e_tokens / e2e_sec, "unit": "tokens/s", "h2d_bytes_per_step": int(h2d),
                "d2h_bytes_per_step": int(d2h), "steps": n_e2e, "ms_per_step": 1e3 * e2e_sec / n_e2e,
                "records_per_s": R * n_e2e * world / e2e_sec},
        "roofline": roof,
        "breakdown_ms_per_step": dict({k: v[0] / steps for k, v in prof.items()}, gemm=g_ms / steps),
        "attention_tflops": a_fl / (a_ms * 1e-3) / 1e12 if a_ms > 0 else None,
        "row_kernels_gbs": r_by / (r_ms * 1e-3) / 1e9 if r_ms > 0 else None,
    }
    if world == 1 and not args.no_cpu_baseline:
        n = seqs_for_tokens(cu, 4000 if workload == "base" else 1500)
        Tc, Sc, dt = oracle_sample_pass(w, desc, rec, win, n, names)
        out["cpu_baseline"] = {"value": Tc / dt, "unit": "tokens/s", "cores": blas_threads(), "kind": "oracle",
                               "sample": "first %d sequences (%d tokens, %d spans) of the workload, %.1f s" % (n, Tc, Sc, dt)}
    return out


def run_stream(args, records=None):
    """BASELINE.json configs[2]: the full synthetic record stream (70,951 records, ~550 MB) in token-budgeted
    batches of whole records; the entity cache persists across batches.  A "step" is one batch (~1 M tokens);
    the timed region is ALL batches of the stream, after 3 warm-up batches run on a scratch cache."""
    import torch
    import paper_2606_15650_b200 as P
    from paper_2606_15650_b200 import sharding, stream
    world, rank, local = dist_setup(args)
    dev = torch.device("cuda", local)
    peaks = measured_peaks()
    t_setup = time.time()
    desc = gen.DESCS["base"]
    n_records = records or 70951
    rec = gen.workload_stream(n_records=n_records, seed=gen.SEED_BASE + 3 + 1000 * rank,
                              n_pool=300000 if n_records >= 20000 else 20000)
    log(f"[rank {rank}] records generated in {time.time() - t_setup:.0f}s: {rec['text'].size / 2**20:.1f} MiB, "
        f"{int(rec['tok_rec_off'][-1])} content tokens, {rec['n_entities']} planted entities")
    win = gen.window_records(rec)
    names = gen.TYPE_NAMES_6
    w = gen.make_weights(desc, gen.SEED_BASE + 2, planted=PLANTED)
    plan = stream.plan_batches(win["win_rec"], win["cu_seqlens"], args.batch_tokens)
    batches = [stream.slice_batch(rec, win, a, b) for a, b in plan]
    T_all = int(win["cu_seqlens"][-1])
    maxT = max(b["token_ids"].size for b in batches)
    maxB = max(b["cu_seqlens"].size - 1 for b in batches)
    max_text = max(b["text"].size for b in batches)
    cap = maxT // 4 + 4096
    out_cap = cap * 32
    ws = P.anon_workspace_bytes(desc, maxT, maxB) + 96 * maxT + 2 * max_text + out_cap + 40 * cap + (128 << 20)
    if args.regex:
        ws += 2 * max_text + 48 * cap + (16 << 20)
    ctx = P.Context(local, workspace_bytes=ws)
    W = P.Weights(ctx, desc, gen.pack_blob(w))
    rx = None
    if args.regex:      # NEXT-4: the hybrid strategy -- regex spans merged into the NER spans before the gather
        from paper_2606_15650_b200 import regex_dfa
        rx = P.Regex(ctx, regex_dfa.compile_patterns(list(enumerate(gen.REGEX_PATTERNS)), 80))
    log(f"[rank {rank}] setup {time.time() - t_setup:.0f}s: {len(batches)} batches, {T_all} window-tokens, "
        f"{len(win['cu_seqlens']) - 1} windows, max batch {maxT} tokens, ws={ws / 2**30:.1f} GiB")

    d = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(dev)
    dbat = [dict(ids=d(b["token_ids"]), cu=d(b["cu_seqlens"]), meta=d(b["meta"]), text=d(b["text"]), ro=d(b["rec_off"]))
            for b in batches]
    labels = torch.zeros(maxT, dtype=torch.int32, device=dev)
    spans = torch.zeros((cap, 4), dtype=torch.int32, device=dev)
    nsp = torch.zeros(1, dtype=torch.int32, device=dev)
    span_bytes = torch.zeros(max_text + 16, dtype=torch.uint8, device=dev)
    span_off = torch.zeros(cap + 1, dtype=torch.int64, device=dev)
    span_type = torch.zeros(cap, dtype=torch.uint8, device=dev)
    out_tokens = torch.zeros(out_cap, dtype=torch.uint8, device=dev)
    out_off = torch.zeros(cap + 1, dtype=torch.int64, device=dev)
    hit = torch.zeros(cap, dtype=torch.uint8, device=dev)
    nsp_host = torch.zeros(1, dtype=torch.int32).pin_memory()
    if rx is not None:
        ner_spans, rx_spans = torch.zeros_like(spans), torch.zeros_like(spans)
        n_ner, n_rx = torch.zeros(1, dtype=torch.int32, device=dev), torch.zeros(1, dtype=torch.int32, device=dev)

    def step(cache, k):
        b = dbat[k]
        T = b["ids"].numel()
        P.anon_ner_forward(ctx, W, b["ids"], b["cu"], None, labels[:T])
        if rx is None:
            P.anon_decode_spans(ctx, labels[:T], b["meta"], desc["num_labels"], spans, nsp)
        else:           # counts stay on the device between decode, scan and merge
            P.anon_decode_spans(ctx, labels[:T], b["meta"], desc["num_labels"], ner_spans, n_ner)
            P.anon_regex_scan(ctx, rx, b["text"], b["ro"], rx_spans, n_rx)
            P.anon_merge_spans(ctx, ner_spans, n_ner, rx_spans, n_rx, spans, nsp)
        nsp_host.copy_(nsp, non_blocking=True)
        rc = ctx.sync()
        if rc:
            raise RuntimeError(f"device status {rc}")
        S = int(nsp_host[0])
        P.anon_gather_spans(ctx, b["text"], b["ro"], spans, S, span_bytes, span_off, span_type)
        P.anon_pseudonymize(ctx, cache, span_bytes, span_off[:S + 1], span_type, KEY, SLUG_LEN, names, out_tokens,
                            out_off[:S + 1], hit)
        # NEXT-1: the records rewritten on the device with every span replaced by its pseudonym (text in -> text out)
        P.anon_splice_records(ctx, b["text"], b["ro"], spans, S, out_tokens, out_off[:S + 1], new_text, new_ro[:b["ro"].numel()])
        return S

    new_text = torch.zeros(max_text + out_cap, dtype=torch.uint8, device=dev)
    new_ro = torch.zeros(max(b["rec_off"].size for b in batches), dtype=torch.int64, device=dev)
    scratch = P.Cache(ctx, 1 << 20, 64 << 20)
    for k in range(min(3, len(batches))):
        step(scratch, k)
    assert ctx.sync() == 0
    scratch.close()
    cache = P.Cache(ctx, 1 << 20, 64 << 20)
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier(world)
    sampler = ClockSampler(gpu_id_for_smi(local)) if rank == 0 else None
    ctx.profile(True)
    ev0.record()
    S_all = 0
    for k in range(len(batches)):
        S_all += step(cache, k)
    ev1.record()
    barrier(world)
    prof, launches = ctx.profile_read()
    ctx.profile(False)
    clocks = sampler.stop() if sampler else None
    sec_local = ev0.elapsed_time(ev1) / 1e3
    st = cache.stats()
    cache.close()
    recs_all, sec = sharding.aggregate_throughput(n_records, sec_local, dev)
    tokens_all, _ = sharding.aggregate_throughput(T_all, sec_local, dev)
    spans_all, _ = sharding.aggregate_throughput(S_all, sec_local, dev)
    del dbat

    # ---- e2e: every batch through anon_pipeline_host from pinned HOST buffers, fresh cache ----
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory().numpy()
    hbat = [dict(ids=pin(b["token_ids"]), cu=pin(b["cu_seqlens"]), meta=pin(b["meta"]), text=pin(b["text"]),
                 ro=pin(b["rec_off"])) for b in batches]
    bufs = dict(spans=torch.zeros((cap, 4), dtype=torch.int32).pin_memory().numpy(),
                out=torch.zeros(out_cap, dtype=torch.uint8).pin_memory().numpy(),
                off=torch.zeros(cap + 1, dtype=torch.int64).pin_memory().numpy(),
                hit=torch.zeros(cap, dtype=torch.uint8).pin_memory().numpy(),
                new_text=torch.zeros(max_text + out_cap, dtype=torch.uint8).pin_memory().numpy(),
                new_ro=torch.zeros(max(b["rec_off"].size for b in batches), dtype=torch.int64).pin_memory().numpy())
    cache2 = P.Cache(ctx, 1 << 20, 64 << 20)
    if rx is not None:
        P.anon_ctx_set_regex(ctx, rx)
    barrier(world)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    h2d = d2h = 0
    hits = out_text_bytes = 0
    e0.record()
    for hb in hbat:
        res = P.anon_pipeline_host(ctx, W, cache2, hb["ids"], hb["cu"], hb["meta"], hb["text"], hb["ro"], KEY, SLUG_LEN,
                                   names, cap, out_cap, want_hit=True, bufs=bufs, want_text=True)     # text in -> text out
        Sh = len(res["spans"])
        hits += int(res["hit"].sum())
        out_text_bytes += int(res["new_text"].size)
        h2d += hb["ids"].nbytes + hb["cu"].nbytes + hb["meta"].nbytes + hb["text"].nbytes + hb["ro"].nbytes
        d2h += Sh * 16 + int(res["out_tokens"].size) + (Sh + 1) * 8 + Sh + 8 + int(res["new_text"].size) + hb["ro"].nbytes
    e1.record()
    barrier(world)
    e2e_recs, e2e_sec = sharding.aggregate_throughput(n_records, e0.elapsed_time(e1) / 1e3, dev)
    st2 = cache2.stats()
    cache2.close(); W.close()
    if rx is not None:
        P.anon_ctx_set_regex(ctx, None)
        rx.close()
    ctx.close()
    del hbat, bufs, labels, spans, span_bytes, span_off, span_type, out_tokens, out_off, hit, new_text, new_ro
    torch.cuda.empty_cache()
    if rank != 0:
        return None, rec
    nb = len(batches)
    roof, g_ms = gemm_rooflines(prof, peaks)
    a_ms, a_fl, _ = prof["attention"]
    r_ms, r_by, _ = prof["row"]
    out = {
        "metric": "records_per_s", "value": recs_all / sec, "unit": "records/s", "n_gpus": world,
        "steps": nb, "warmup": min(3, nb), "ms_per_step": 1e3 * sec / nb, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "bf16", "data": "synthetic",
        "config": {"workload": "BASELINE.json configs[2]: %d synthetic records, %.1f MiB of text, %d windows (510+2, overlap 128), "
                               "%d window-tokens, Zipf(1.1) entities; batches of whole records, <= %d tokens"
                               % (n_records, rec["text"].size / 2**20, len(win["cu_seqlens"]) - 1, T_all, args.batch_tokens),
                   "batches": nb, "weights": "W2 planted-detector (deep variant), seeded random-init", "slug_len": SLUG_LEN,
                   "splice": "records rewritten on the device (anon_splice_records) inside the timed region",
                   "regex": ("hybrid detection: DFA scan of %d patterns over the batch text + regex/NER span merge inside the "
                             "timed region (NEXT-4)" % len(gen.REGEX_PATTERNS)) if rx is not None else "off (--regex enables NEXT-4)",
                   "spans": S_all, "planted_entities": int(rec["n_entities"]), "unique_entities": st["n_unique"],
                   "cache_hit_rate": st["n_hits"] / max(st["n_lookups"], 1),
                   "l2": "inputs larger than L2 (each batch streams ~20 GB of activations through HBM)"},
        "seconds_whole_stream": sec, "tokens_per_s": tokens_all / sec, "spans_per_s": spans_all / sec,
        "kb_per_s": rec["text"].size / 1024.0 * world / sec,
        "clocks": clocks, "gpu_launches": launches,
        "e2e": {"value": e2e_recs / e2e_sec, "unit": "records/s", "h2d_bytes_per_step": int(h2d // nb),
                "d2h_bytes_per_step": int(d2h // nb), "steps": nb, "seconds_whole_stream": e2e_sec,
                "tokens_per_s": T_all * world / e2e_sec, "kb_per_s": rec["text"].size / 1024.0 * world / e2e_sec,
                "cache_hit_rate": st2["n_hits"] / max(st2["n_lookups"], 1),
                "call": "anon_pipeline_host_text: records in, rewritten records out", "rewritten_text_bytes": out_text_bytes},
        "roofline": roof,
        "breakdown_ms_per_step": dict({k: v[0] / nb for k, v in prof.items()}, gemm=g_ms / nb),
        "attention_tflops": a_fl / (a_ms * 1e-3) / 1e12 if a_ms > 0 else None,
        "row_kernels_gbs": r_by / (r_ms * 1e-3) / 1e9 if r_ms > 0 else None,
    }
    if world == 1 and not args.no_cpu_baseline:
        n = seqs_for_tokens(win["cu_seqlens"], 4000)
        Tc, Sc, dt = oracle_sample_pass(w, desc, rec, win, n, names)
        out["cpu_baseline"] = {"value": n_records * (Tc / dt) / T_all, "unit": "records/s", "cores": blas_threads(),
                               "kind": "oracle",
                               "sample": "first %d windows (%d tokens, %d spans) of the stream in %.1f s = %.0f tokens/s, "
                                         "scaled by tokens per record" % (n, Tc, Sc, dt, Tc / dt)}
    return out, rec


def pseudonym_alg_bytes(span_bytes, S, out_bytes):
    """Algorithmic bytes of anon_pseudonymize: span bytes once for the hash + once for the compare against the
    stored key, 16 B of offsets, one 32 B slot sector, hit / uid / type (10 B), the token written and its 8 B offset."""
    return 2 * span_bytes + 16 * S + 32 * S + 10 * S + out_bytes + 8 * S


def run_pseudonym(args, records=None, steps=None, warmup=None):
    """BASELINE.json configs[4]: 50 M spans Zipf(1.1) over 2 M strings -> dedup + HMAC + write-back."""
    import torch
    import paper_2606_15650_b200 as P
    from paper_2606_15650_b200 import sharding
    steps = steps or args.steps
    warmup = args.warmup if warmup is None else warmup
    world, rank, local = dist_setup(args)
    dev = torch.device("cuda", local)
    peaks = measured_peaks()
    n_unique, n_draws = (records or 2_000_000), (records or 2_000_000) * 25
    t0 = time.time()
    data, off, types, key, _ = gen.spans_zipf(n_unique, n_draws, 7, 128, 6, gen.SEED_BASE + 5 + 1000 * rank)
    log(f"[rank {rank}] generated {n_draws} spans, {data.size / 1e9:.2f} GB in {time.time() - t0:.0f}s")
    S = n_draws
    ctx = P.Context(local, workspace_bytes=S * 9 + (S // 2048 + 2) * 24 + (64 << 20))
    cache = P.Cache(ctx, n_unique, int(n_unique * 70) + (1 << 20))
    d_bytes, d_off, d_type = (torch.from_numpy(a).to(dev) for a in (data, off, types))
    out_cap = S * (3 + 13 + SLUG_LEN)
    out = torch.zeros(out_cap, dtype=torch.uint8, device=dev)
    out_off = torch.zeros(S + 1, dtype=torch.int64, device=dev)
    hit = torch.zeros(S, dtype=torch.uint8, device=dev)
    uid = torch.zeros(S, dtype=torch.int64, device=dev)
    kb = key.tobytes()

    def step():
        cache.clear()
        P.anon_pseudonymize(ctx, cache, d_bytes, d_off, d_type, kb, SLUG_LEN, gen.TYPE_NAMES_6, out, out_off, hit, uid)
    for _ in range(warmup):
        step()
    assert ctx.sync() == 0
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier(world)
    sampler = ClockSampler(gpu_id_for_smi(local)) if rank == 0 else None
    ctx.profile(True)
    ev0.record()
    for _ in range(steps):
        step()
    ev1.record()
    barrier(world)
    prof, launches = ctx.profile_read()
    ctx.profile(False)
    clocks = sampler.stop() if sampler else None
    spans_all, sec = sharding.aggregate_throughput(S * steps, ev0.elapsed_time(ev1) / 1e3, dev)
    st = cache.stats()
    out_bytes = int(out_off[S].item())
    alg = pseudonym_alg_bytes(data.size, S, out_bytes)

    # ---- e2e: span bytes / offsets / types in pinned HOST buffers -> H2D -> anon_pseudonymize -> D2H of tokens, offsets, hit ----
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
    h_bytes, h_off, h_type = pin(data), pin(off), pin(types)
    h_out = torch.zeros(out_bytes, dtype=torch.uint8).pin_memory()
    h_out_off = torch.zeros(S + 1, dtype=torch.int64).pin_memory()
    h_hit = torch.zeros(S, dtype=torch.uint8).pin_memory()

    def step_host():
        cache.clear()
        d_bytes.copy_(h_bytes, non_blocking=True); d_off.copy_(h_off, non_blocking=True); d_type.copy_(h_type, non_blocking=True)
        P.anon_pseudonymize(ctx, cache, d_bytes, d_off, d_type, kb, SLUG_LEN, gen.TYPE_NAMES_6, out, out_off, hit, None)
        h_out.copy_(out[:out_bytes], non_blocking=True); h_out_off.copy_(out_off, non_blocking=True); h_hit.copy_(hit, non_blocking=True)
    step_host()
    barrier(world)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    n_e2e = max(1, min(steps, 3))
    e0.record()
    for _ in range(n_e2e):
        step_host()
    e1.record()
    barrier(world)
    e2e_spans, e2e_sec = sharding.aggregate_throughput(S * n_e2e, e0.elapsed_time(e1) / 1e3, dev)
    assert ctx.sync() == 0
    h2d, d2h = data.nbytes + off.nbytes + types.nbytes, out_bytes + (S + 1) * 8 + S
    cache.close(); ctx.close()
    del d_bytes, d_off, d_type, out, out_off, hit, uid, h_bytes, h_off, h_type, h_out, h_out_off, h_hit
    torch.cuda.empty_cache()
    if rank != 0:
        return None
    ms = prof["pseudonymize"][0] / steps
    res = {"metric": "pseudonym_spans_per_s", "value": spans_all / sec, "unit": "spans/s", "n_gpus": world,
           "steps": steps, "warmup": warmup, "ms_per_step": 1e3 * sec / steps, "higher_is_better": True,
           "scaling": "weak", "vs_baseline": None, "dtype": "u32", "data": "synthetic",
           "config": {"workload": "BASELINE.json configs[4]: %d spans of 7-128 B, Zipf(1.1) over %d strings" % (S, n_unique),
                      "unique_found": st["n_unique"], "hit_rate": st["n_hits"] / max(st["n_lookups"], 1),
                      "l2": "inputs larger than L2 (%.1f GB of span bytes)" % (data.size / 1e9)},
           "clocks": clocks, "gpu_launches": launches,
           "e2e": {"value": e2e_spans / e2e_sec, "unit": "spans/s", "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h),
                   "steps": n_e2e, "ms_per_step": 1e3 * e2e_sec / n_e2e,
                   "call": "pinned host span CSR -> H2D -> anon_pseudonymize -> D2H of tokens, offsets, hit flags"},
           "roofline": {"bound": "hbm", "kernel": "anon_pseudonymize (probe + classify scan + insert/HMAC + emit)",
                        "achieved": alg / (ms * 1e-3) / 1e9, "peak": peaks["hbm_gbs"], "unit": "GB/s",
                        "frac": alg / (ms * 1e-3) / 1e9 / peaks["hbm_gbs"], "traffic": None,
                        "algorithmic_bytes_per_step": int(alg), "avg_launch_ms": ms,
                        "peak_source": "MEASURED_PEAKS.json hbm_gbs (%s)" % peaks["source"]}}
    if world == 1 and not args.no_cpu_baseline:
        from oracle import crypto
        oc = crypto.Cache(1 << 22)
        t0 = time.perf_counter()
        oc.pseudonymize(data, off, types, kb, SLUG_LEN, gen.TYPE_NAMES_6)
        dt = time.perf_counter() - t0
        oc.close()
        res["cpu_baseline"] = {"value": S / dt, "unit": "spans/s", "cores": 1, "kind": "oracle",
                               "sample": "the FULL workload (%d spans, %d unique) through oracle/anon_oracle.c, one thread, %.1f s" % (S, st["n_unique"], dt)}
    return res


FIELD_TYPE = 2          # NEXT-2: every field span carries one fixed type (the schema names the field)


def oracle_fields_pass(rec, n_records):
    """The oracle over the first n_records records of the field workload: gather + dedup / HMAC / write-back + splice."""
    from oracle import crypto, decode
    ro = rec["rec_off"][:n_records + 1]
    text = rec["text"][:int(ro[-1])]
    spans = gen.field_spans(rec, FIELD_TYPE)
    spans = spans[spans[:, 0] < n_records]
    sp = [tuple(int(v) for v in s) for s in spans]
    t0 = time.perf_counter()
    sb, so = decode.gather_spans(text, ro, sp)
    oc = crypto.Cache(1 << 20)
    w = oc.pseudonymize(sb, so, spans[:, 3].astype(np.uint8), KEY, SLUG_LEN, gen.TYPE_NAMES_6)
    decode.splice_records(text, ro, sp, w["out_tokens"], w["out_offsets"])
    dt = time.perf_counter() - t0
    oc.close()
    return text.size, len(sp), dt


def run_fields(args, rec=None, records=None, steps=None, warmup=None):
    """S8f NEXT-2: caller-supplied field spans with a fixed type over the configs[2] record text ->
    anon_gather_spans -> anon_pseudonymize -> anon_splice_records.  No encoder kernel runs.  Unit: KB of record text per second
    (the paper's unit for this path: 34,341 KB/s for D2-CSV on its machine -- context, not the target)."""
    import torch
    import paper_2606_15650_b200 as P
    from paper_2606_15650_b200 import sharding
    steps = steps or args.steps
    warmup = args.warmup if warmup is None else warmup
    world, rank, local = dist_setup(args)
    dev = torch.device("cuda", local)
    peaks = measured_peaks()
    if rec is None:
        n_records = records or 70951
        rec = gen.workload_stream(n_records=n_records, seed=gen.SEED_BASE + 3 + 1000 * rank, n_pool=300000 if n_records >= 20000 else 20000)
    text, ro = rec["text"], rec["rec_off"]
    spans = gen.field_spans(rec, FIELD_TYPE)
    S, R = int(spans.shape[0]), int(ro.size - 1)
    sb_total = int((spans[:, 2] - spans[:, 1]).sum())
    ctx = P.Context(local, workspace_bytes=(64 << 20) + 64 * S)
    cache = P.Cache(ctx, 1 << 20, 64 << 20)
    d = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(dev)
    d_text, d_ro, d_spans = d(text), d(ro), d(spans)
    span_bytes = torch.zeros(sb_total + 16, dtype=torch.uint8, device=dev)
    span_off = torch.zeros(S + 1, dtype=torch.int64, device=dev)
    span_type = torch.zeros(S, dtype=torch.uint8, device=dev)
    out_cap = S * (3 + 13 + SLUG_LEN)
    out = torch.zeros(out_cap, dtype=torch.uint8, device=dev)
    out_off = torch.zeros(S + 1, dtype=torch.int64, device=dev)
    hit = torch.zeros(S, dtype=torch.uint8, device=dev)
    new_text = torch.zeros(text.size + out_cap, dtype=torch.uint8, device=dev)
    new_ro = torch.zeros(R + 1, dtype=torch.int64, device=dev)

    def step():
        cache.clear()
        P.anon_gather_spans(ctx, d_text, d_ro, d_spans, S, span_bytes, span_off, span_type)
        P.anon_pseudonymize(ctx, cache, span_bytes, span_off, span_type, KEY, SLUG_LEN, gen.TYPE_NAMES_6, out, out_off, hit)
        P.anon_splice_records(ctx, d_text, d_ro, d_spans, S, out, out_off, new_text, new_ro)
    for _ in range(warmup):
        step()
    assert ctx.sync() == 0
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier(world)
    sampler = ClockSampler(gpu_id_for_smi(local)) if rank == 0 else None
    ctx.profile(True)
    ev0.record()
    for _ in range(steps):
        step()
    ev1.record()
    barrier(world)
    prof, launches = ctx.profile_read()
    ctx.profile(False)
    clocks = sampler.stop() if sampler else None
    bytes_all, sec = sharding.aggregate_throughput(text.size * steps, ev0.elapsed_time(ev1) / 1e3, dev)
    st = cache.stats()
    out_bytes = int(out_off[S].item())
    new_bytes = int(new_ro[R].item())
    alg = (16 * S + 2 * sb_total + 8 * S) + pseudonym_alg_bytes(sb_total, S, out_bytes) + (text.size + new_bytes + out_bytes + 24 * S)

    # ---- e2e: text, record offsets and field spans in pinned HOST buffers; the rewritten text comes back to the host ----
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
    h_text, h_ro, h_spans = pin(text), pin(ro), pin(spans)
    h_new_text = torch.zeros(text.size + out_cap, dtype=torch.uint8).pin_memory()
    h_new_ro = torch.zeros(R + 1, dtype=torch.int64).pin_memory()

    def step_host():
        d_text.copy_(h_text, non_blocking=True); d_ro.copy_(h_ro, non_blocking=True); d_spans.copy_(h_spans, non_blocking=True)
        step()
        h_new_ro.copy_(new_ro, non_blocking=True)
        if ctx.sync():
            raise RuntimeError("device status")
        n = int(h_new_ro[R])
        h_new_text[:n].copy_(new_text[:n], non_blocking=True)
        return n
    step_host()
    barrier(world)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    n_e2e = max(1, min(steps, 3))
    e0.record()
    for _ in range(n_e2e):
        n_out = step_host()
    e1.record()
    barrier(world)
    e2e_bytes, e2e_sec = sharding.aggregate_throughput(text.size * n_e2e, e0.elapsed_time(e1) / 1e3, dev)
    h2d, d2h = text.nbytes + ro.nbytes + spans.nbytes, n_out + (R + 1) * 8
    cache.close(); ctx.close()
    del d_text, d_ro, d_spans, span_bytes, span_off, span_type, out, out_off, hit, new_text, new_ro, h_text, h_new_text
    torch.cuda.empty_cache()
    if rank != 0:
        return None
    ms = 1e3 * sec / steps
    res = {"metric": "field_path_kb_per_s", "value": bytes_all / 1024.0 / sec, "unit": "KB/s", "n_gpus": world,
           "steps": steps, "warmup": warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
           "dtype": "u32", "data": "synthetic",
           "config": {"workload": "S8f NEXT-2 on the BASELINE.json configs[2] records: %d records, %.1f MiB of text, %d field spans of one "
                                  "fixed type (%s), no NER" % (R, text.size / 2**20, S, gen.TYPE_NAMES_6[FIELD_TYPE]),
                      "unique_entities": st["n_unique"], "cache_hit_rate": st["n_hits"] / max(st["n_lookups"], 1),
                      "l2": "inputs larger than L2 (%.0f MB of text per step)" % (text.size / 1e6),
                      "calls": "anon_gather_spans -> anon_pseudonymize -> anon_splice_records"},
           "spans_per_s": S * steps * world / sec, "records_per_s": R * steps * world / sec,
           "clocks": clocks, "gpu_launches": launches,
           "e2e": {"value": e2e_bytes / 1024.0 / e2e_sec, "unit": "KB/s", "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h),
                   "steps": n_e2e, "ms_per_step": 1e3 * e2e_sec / n_e2e, "records_per_s": R * n_e2e * world / e2e_sec,
                   "call": "pinned host text + field spans -> H2D -> gather / pseudonymize / splice -> D2H of the rewritten text"},
           "roofline": {"bound": "hbm", "kernel": "field path: gather + pseudonymize + splice (all launches of the step)",
                        "achieved": alg / (ms * 1e-3) / 1e9, "peak": peaks["hbm_gbs"], "unit": "GB/s",
                        "frac": alg / (ms * 1e-3) / 1e9 / peaks["hbm_gbs"], "traffic": None, "algorithmic_bytes_per_step": int(alg),
                        "peak_source": "MEASURED_PEAKS.json hbm_gbs (%s)" % peaks["source"]},
           "breakdown_ms_per_step": {k: prof[k][0] / steps for k in ("decode", "pseudonymize")}}
    if world == 1 and not args.no_cpu_baseline:
        nb, ns, dt = oracle_fields_pass(rec, min(R, 1500))
        res["cpu_baseline"] = {"value": nb / 1024.0 / dt, "unit": "KB/s", "cores": 1, "kind": "oracle",
                               "sample": "first %d records (%.1f MiB, %d field spans) in %.1f s" % (min(R, 1500), nb / 2**20, ns, dt)}
    return res


def free_port():
    with socket.socket(socket.AF_INET, socket.SOCK_STREAM) as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="base", choices=["base", "large", "stream", "pseudonym", "fields", "modern"])
    ap.add_argument("--records", type=int, default=None, help="override the number of records / sequences / strings")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--headline-only", action="store_true", help="only the timed configs[1] line, none of the extra legs")
    ap.add_argument("--extra-budget-s", type=float, default=840.0,
                    help="wall-clock budget of the whole run; an extra leg that would not fit is skipped and says so")
    ap.add_argument("--batch-tokens", type=int, default=1 << 20, help="stream workload: token budget per batch")
    ap.add_argument("--regex", action="store_true", help="stream workload: also run the regex detector and merge its spans (NEXT-4)")
    args = ap.parse_args()
    world_env = os.environ.get("WORLD_SIZE")
    if args.gpus > 1 and world_env is None:
        # `python bench.py --gpus N`: become N ranks, one per GPU, under torchrun on this node (S8e)
        cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
               "--master-addr", "127.0.0.1", "--master-port", str(free_port()), os.path.abspath(__file__)] + sys.argv[1:]
        log("bench.py: re-executing under torchrun:", " ".join(cmd))
        os.environ.setdefault("NCCL_DEBUG", "WARN")
        os.execv(sys.executable, cmd)
    if world_env is not None and int(world_env) != args.gpus:
        raise SystemExit(f"bench.py: --gpus {args.gpus} does not match WORLD_SIZE={world_env}")
    if args.warmup < 3 and args.impl == "ours":
        log("note: timing rules ask for >= 3 warm-up steps")
    if args.impl == "reference":
        return run_reference(args)
    world = int(world_env or "1")
    if args.workload == "pseudonym":
        out = run_pseudonym(args, records=args.records)
    elif args.workload == "stream":
        out, _ = run_stream(args, records=args.records)
    elif args.workload == "fields":
        out = run_fields(args, records=args.records)
    else:
        out = run_encoder(args, records=args.records)
    if out is None:            # ranks > 0
        return
    if args.workload == "base" and args.records is None and world == 1 and not args.headline_only:
        # the headline configs of BASELINE.json next to the timed configs[1] line, each in its own timed region
        rec = None
        est = {"stream": 260, "pseudonym": 170, "large": 110, "fields": 60}           # seconds each leg needs on the box
        for name in ("stream", "pseudonym", "large", "fields"):
            left = args.extra_budget_s - (time.time() - T_START)
            need = est[name] + (80 if name == "fields" and rec is None else 0)
            if left < need:
                out[name] = {"skipped": "time budget: %.0f s left, this leg needs about %d s (--extra-budget-s)" % (left, need)}
                log(f"[extra] {name}: skipped ({left:.0f}s left)")
                continue
            t0 = time.time()
            try:
                if name == "stream":
                    out[name], rec = run_stream(args)
                elif name == "pseudonym":
                    out[name] = run_pseudonym(args, steps=5, warmup=3)
                elif name == "large":
                    out[name] = run_encoder(args, workload="large", steps=3, warmup=3, e2e_steps=2)
                else:
                    out[name] = run_fields(args, rec=rec, steps=5, warmup=3)
            except Exception as e:     # an extra leg must never cost the timed line
                out[name] = {"error": "%s: %s" % (type(e).__name__, e)}
            log(f"[extra] {name}: {time.time() - t0:.0f}s")
        out["wall_s_total"] = time.time() - T_START
    print(json.dumps(out), flush=True)


if __name__ == "__main__":
    main()
