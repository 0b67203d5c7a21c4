"""Per-kernel roofline measurements through the C ABI (the single-kernel entry points of include/anonshield.h).

    python kernel_bench.py [--tokens 262144] [--hidden 768] [--spans 8000000]

Times, with CUDA events on the context's stream after warm-up: the four encoder GEMM shapes (QKV, out-proj+residual,
FFN1+GELU, FFN2+residual) against cuBLAS (torch.matmul, no epilogue -- context, not the product), the varlen
attention kernel on a lognormal length mix and at n = 512, the HMAC-SHA256 kernel with dedup disabled
(anon_hmac_spans; SURVEY.md §8(d) c5 "HMAC-only run"), and the DFA regex scan (NEXT-4) over 400 MB of record text.  Prints one JSON object; inputs are seeded and larger than
L2 where the kernel is memory-bound.  Peaks: MEASURED_PEAKS.json (else the B200_PROFILING.md fallback).
"""
import argparse
import json
import os
import subprocess
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def _peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            d = json.load(f)
        return d["hbm_gbs"], d["bf16_tflops"], "measured"
    return 6650.0, 1590.0, "fallback"


def _att_prof(P):
    """Cycles per 128 x 64 chunk in each wait / phase of the MMA issuer and of two softmax warps of virtual CTA 0, from the clock64
    counters an ATT_PROF build of attention_bf16.cu keeps (the counters themselves cost ~40-60 cycles per reading)."""
    import ctypes
    from paper_2606_15650_b200 import binding
    lib = binding.lib()
    if not hasattr(lib, "anon_debug_att_prof"):
        raise SystemExit("--att-prof: rebuild with ANON_NVCC_EXTRA=-DATT_PROF=1")
    buf = (ctypes.c_ulonglong * 64)()
    if lib.anon_debug_att_prof(buf) != 0:
        raise SystemExit("--att-prof: cudaMemcpyFromSymbol failed")
    v = list(buf)
    names = {"mma_issuer": ["wait_s_free", "wait_q_full", "wait_k_full", "issue_qk", "wait_v_full", "wait_p_full", "wait_o_empty", "issue_pv"],
             "softmax_warp": ["wait_s_full", "tmem_ld+arrive", "max(+rescale)", "exp+sum+pack", "wait_pv_done", "tmem_st+arrive", "finalize"]}
    out = {}
    for off, key, tag in ((0, "mma_issuer", "mma_issuer"), (16, "softmax_warp", "softmax_warp_a"), (32, "softmax_warp", "softmax_warp_b")):
        ch = max(1, v[off + 9])
        out[tag] = {"chunks": v[off + 9], "total": round(v[off + 8] / ch, 1), **{n: round(v[off + i] / ch, 1) for i, n in enumerate(names[key])}}
    return out


def main():
    import torch
    import paper_2606_15650_b200 as P
    from harness import gen
    ap = argparse.ArgumentParser()
    ap.add_argument("--tokens", type=int, default=262144)
    ap.add_argument("--hidden", type=int, default=768)
    ap.add_argument("--spans", type=int, default=8_000_000)
    ap.add_argument("--iters", type=int, default=10)
    ap.add_argument("--regex-records", type=int, default=2000)
    ap.add_argument("--regex-mb", type=float, default=400.0)
    ap.add_argument("--att-prof", action="store_true",
                    help="print the attention kernel's clock64 counters after each attention run (needs a library built with "
                         "ANON_NVCC_EXTRA=-DATT_PROF=1, which exports anon_debug_att_prof)")
    ap.add_argument("--only", default="", help="comma list out of gemm,attention,hmac,regex (default: all); the issue-rate peaks always run")
    args = ap.parse_args()
    only = set(x for x in args.only.split(",") if x)
    want = lambda name: not only or name in only
    if not torch.cuda.is_available():
        raise SystemExit("kernel_bench: no CUDA device (the hot path has no CPU fallback)")
    dev = torch.device("cuda", 0)
    M, H = args.tokens, args.hidden
    F = 4 * H
    hbm, tf_peak, src = _peaks()
    ctx = P.Context(0, workspace_bytes=256 << 20)

    clocks_after = []          # SM clock right after each timed loop, in call order

    def sm_mhz():
        try:
            return float(subprocess.check_output(["nvidia-smi", "-i", "0", "--query-gpu=clocks.sm", "--format=csv,noheader,nounits"],
                                                 text=True).strip().splitlines()[0])
        except Exception:
            return None

    def timeit(fn, n=args.iters, warm=3):
        # every kernel is timed ALONE: two seconds of idle first, so that the clock the power-capped GEMM loops leave behind
        # (1.0-1.3 GHz) does not carry into the next measurement; the clock right after the loop is reported with each number
        torch.cuda.synchronize()
        time.sleep(2.0)
        for _ in range(warm):
            fn()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(n):
            fn()
        e1.record()
        torch.cuda.synchronize()
        clocks_after.append(sm_mhz())
        return e0.elapsed_time(e1) / n

    res = {"peaks": {"hbm_gbs": hbm, "bf16_tflops_burst": tf_peak, "source": src}, "tokens": M, "hidden": H}
    # measured issue-rate peaks (anon_microbench): thread-ops/s of the integer-ALU pipe and of MUFU ex2, and the lanes/clk/SM
    # they amount to at the clock nvidia-smi reports right after the run ("record which of 64 / 128")
    sms = torch.cuda.get_device_properties(0).multi_processor_count
    names = {0: "lop3+shf+iadd3 mix (ALU + FMA pipes)", 1: "lop3", 2: "shf", 3: "iadd3", 4: "mufu_ex2"}
    mb = {}
    for mode, nm in names.items():
        P.anon_microbench(ctx, mode, 256)
        ops, ms = P.anon_microbench(ctx, mode, 4096)
        try:
            mhz = float(subprocess.check_output(["nvidia-smi", "-i", "0", "--query-gpu=clocks.sm", "--format=csv,noheader,nounits"],
                                                text=True).strip().splitlines()[0])
        except Exception:
            mhz = None
        mb[nm] = {"thread_ops_per_s": ops, "kernel_ms": ms, "sm_mhz_after": mhz,
                  "lanes_per_clk_per_sm": ops / (sms * mhz * 1e6) if mhz else None}
    res["issue_rate_peaks"] = mb
    alu_peak_measured = min(mb["lop3"]["thread_ops_per_s"], mb["shf"]["thread_ops_per_s"], mb["iadd3"]["thread_ops_per_s"])
    exp_peak_measured = mb["mufu_ex2"]["thread_ops_per_s"]
    g = torch.Generator(device=dev).manual_seed(260615650)
    for name, N, K, epi in ([("qkv", 3 * H, H, 0), ("out_residual", H, H, 2), ("ffn1_gelu", F, H, 1), ("ffn2_residual", H, F, 2)] if want("gemm") else []):
        A = (torch.randn(M, K, device=dev, generator=g) * 0.5).to(torch.bfloat16)
        W = (torch.randn(N, K, device=dev, generator=g) * 0.02).to(torch.bfloat16)
        bias = torch.randn(N, device=dev, generator=g) * 0.02
        resid = torch.randn(M, N, device=dev, generator=g) if epi == 2 else None
        C = torch.empty(M, N, device=dev, dtype=torch.float32 if epi == 2 else torch.bfloat16)
        ms = timeit(lambda: P.anon_gemm_bf16(ctx, A, W, bias, resid, C, epi))
        ms_ref = timeit(lambda: torch.matmul(A, W.t()))
        fl = 2.0 * M * N * K
        byts = M * K * 2 + N * K * 2 + M * N * (8 if epi == 2 else 2)
        res[name] = {"M": M, "N": N, "K": K, "ms": ms, "sm_mhz_after": clocks_after[-2], "tflops": fl / ms / 1e9, "frac_of_bf16_peak": fl / ms / 1e9 / tf_peak,
                     "algorithmic_gbs": byts / ms / 1e6, "frac_of_hbm_peak": byts / ms / 1e6 / hbm,
                     "cublas_no_epilogue_ms": ms_ref, "cublas_no_epilogue_tflops": fl / ms_ref / 1e9}
        del A, W, C, resid

    rng = np.random.default_rng(1)
    for name, lens in ([("attention_lognormal", np.clip(np.round(rng.lognormal(np.log(200), 0.75, 100000)), 10, 512)),
                        ("attention_n512", np.full(M // 512 + 1, 512))] if want("attention") else []):
        lens = lens.astype(np.int64)
        cu = np.zeros(len(lens) + 1, np.int64)
        cu[1:] = np.cumsum(lens)
        B = max(1, int(np.searchsorted(cu, M, side="right")) - 1)
        cu = cu[:B + 1].astype(np.int32)
        T = int(cu[-1])
        qkv = torch.randn(T, 3 * H, device=dev, generator=g).to(torch.bfloat16)
        out = torch.empty(T, H, device=dev, dtype=torch.bfloat16)
        d_cu = torch.from_numpy(cu).to(dev)
        ms = timeit(lambda: P.anon_attention(ctx, qkv, d_cu, cu, H, H // 64, 1, out))
        prof = _att_prof(P) if args.att_prof else None
        n2 = float((lens[:B].astype(np.float64) ** 2).sum())
        res[name] = {"tokens": T, "sequences": B, "ms": ms, "sm_mhz_after": clocks_after[-1], "tflops": 4.0 * n2 * H / ms / 1e9,
                     "exp_per_s": n2 * (H // 64) / ms * 1e3, "frac_of_measured_exp_peak": n2 * (H // 64) / ms * 1e3 / exp_peak_measured,
                     "frac_of_bf16_burst_peak": 4.0 * n2 * H / ms / 1e9 / tf_peak, "algorithmic_gbs": T * H * 2 * 4 / ms / 1e6}
        if prof:
            res[name]["cycles_per_chunk"] = prof
        # NEXT-3: the same inputs through the banded kernel (window 128): a query sees at most 129 keys
        ms = timeit(lambda: P.anon_attention_local(ctx, qkv, d_cu, cu, H, H // 64, 1, 128, out))
        ln = lens[:B].astype(np.float64)
        vis = float(sum(np.minimum(np.arange(n) + 64, n - 1).sum() - np.maximum(np.arange(n) - 64, 0).sum() + n for n in lens[:B]))
        res[name + "_window128"] = {"tokens": T, "sequences": B, "ms": ms, "visible_pairs": vis, "tflops": 4.0 * vis * H / ms / 1e9,
                                    "exp_per_s": vis * (H // 64) / ms * 1e3, "algorithmic_gbs": T * H * 2 * 4 / ms / 1e6}
        del qkv, out

    if want("hmac"):
        # HMAC-SHA256 with dedup disabled: integer-ALU bound (K10)
        S = args.spans
        data, off, types, key, _ = gen.spans_zipf(200_000, S, 7, 128, 6, gen.SEED_BASE + 5)
        d_bytes, d_off = torch.from_numpy(data).to(dev), torch.from_numpy(off).to(dev)
        dig = torch.empty((S, 32), dtype=torch.uint8, device=dev)
        kb = key.tobytes()
        ms = timeit(lambda: P.anon_hmac_spans(ctx, d_bytes, d_off, kb, dig), n=5)
        lens = np.diff(off)
        comp = float(((lens + 9 + 63) // 64 + 1).sum())
        # ALU-pipe instructions per SHA-256 compression counted in the SASS of hmac_spans_kernel (cuobjdump: 1,363 SHF + 774 LOP3
        # + 531 IADD3 over the two inlined compressions = 1,334 each; another 190 IMAD go to the FMA pipe).  ALU-pipe peak
        # (DESIGN.md section 6): 148 SMs x 64 lanes/clk x 1.965 GHz = 18.6 T lane-instructions/s.
        alu_per_comp, alu_peak = 1334.0, alu_peak_measured          # peak = the measured LOP3 / SHF / IADD3 rate (the slowest of the three)
        res["hmac_sha256_no_dedup"] = {"spans": S, "ms": ms, "hmac_per_s": S / ms * 1e3, "compressions_per_s": comp / ms * 1e3,
                                       "bytes_per_s_gb": (data.size + S * 40) / ms / 1e6,
                                       "roofline": {"bound": "alu", "achieved": comp / ms * 1e3 * alu_per_comp / 1e12, "peak": alu_peak / 1e12,
                                                    "unit": "T ALU-pipe instr/s", "frac": comp / ms * 1e3 * alu_per_comp / alu_peak,
                                                    "peak_source": "anon_microbench modes 1-3 (measured on this box)",
                                                    "derived_peak_148x64x1.965GHz": 148 * 64 * 1.965e9 / 1e12}}

    if want("regex"):
        # NEXT-4: DFA regex scan over record text (HBM-bound; algorithmic traffic = 1 B per text byte read + 16 B per span written)
        from paper_2606_15650_b200 import regex_dfa
        rec = gen.workload_stream(n_records=args.regex_records, n_pool=50000)
        reps = max(1, int(args.regex_mb * 1e6 / rec["text"].size))
        text = np.tile(rec["text"], reps)
        sizes = np.tile(np.diff(rec["rec_off"]), reps)
        roff = np.zeros(sizes.size + 1, np.int64)
        roff[1:] = np.cumsum(sizes)
        blob = regex_dfa.compile_patterns(list(enumerate(gen.REGEX_PATTERNS)), 80)
        d_text, d_roff = torch.from_numpy(text).to(dev), torch.from_numpy(roff).to(dev)
        cap = text.size // 40
        spans = torch.empty((cap, 4), dtype=torch.int32, device=dev)
        num = torch.zeros(1, dtype=torch.int32, device=dev)
        ctx2 = P.Context(0, workspace_bytes=int(text.size * 2.2) + (64 << 20))
        rx2 = P.Regex(ctx2, blob)
        ms = timeit(lambda: P.anon_regex_scan(ctx2, rx2, d_text, d_roff, spans, num), n=5)
        assert ctx2.sync() == 0
        nsp = int(num.item())
        byts = text.size + 16.0 * nsp + 8.0 * roff.size
        res["regex_scan"] = {"text_bytes": int(text.size), "records": int(sizes.size), "spans": nsp, "ms": ms,
                             "text_gb_per_s": text.size / ms / 1e6,
                             "roofline": {"bound": "hbm", "achieved": byts / ms / 1e6, "peak": hbm, "unit": "GB/s", "frac": byts / ms / 1e6 / hbm}}
        rx2.close(); ctx2.close()
    print(json.dumps(res, indent=1))
    ctx.close()


if __name__ == "__main__":
    main()
