"""Thin ctypes binding of include/anonshield.h: argument marshalling only -- every step of the hot path runs
in the CUDA kernels of libanonshield.so.  Device buffers are torch tensors (PyTorch is used for device
memory and streams only); their `data_ptr()` goes straight through the C ABI.

There is no CPU fallback: if the library cannot be built/loaded, importing the symbols raises; if no CUDA
device is present, `Context()` raises AnonError(ANON_ERR_CUDA).
"""
import ctypes
import os

import numpy as np

from . import build as _build

OK, ERR_INVALID_ARG, ERR_UNSUPPORTED, ERR_CAPACITY, ERR_KEY_MISMATCH, ERR_CUDA, ERR_OOM = 0, -1, -2, -3, -4, -5, -6


class ModelDesc(ctypes.Structure):
    _fields_ = [("layers", ctypes.c_int32), ("hidden", ctypes.c_int32), ("heads", ctypes.c_int32),
                ("ffn", ctypes.c_int32), ("vocab", ctypes.c_int32), ("num_labels", ctypes.c_int32),
                ("max_pos", ctypes.c_int32), ("ln_eps", ctypes.c_float), ("dtype", ctypes.c_int32),
                ("arch", ctypes.c_int32), ("local_window", ctypes.c_int32), ("global_every", ctypes.c_int32),
                ("rope_theta_global", ctypes.c_float), ("rope_theta_local", ctypes.c_float)]

    @classmethod
    def from_dict(cls, d):
        return cls(d["layers"], d["hidden"], d["heads"], d["ffn"], d["vocab"], d["num_labels"], d["max_pos"],
                   d["ln_eps"], d["dtype"], d.get("arch", 0), d.get("local_window", 0), d.get("global_every", 1),
                   d.get("rope_theta_global", 0.0), d.get("rope_theta_local", 0.0))


class AnonError(RuntimeError):
    def __init__(self, code, where, detail=""):
        self.code = code
        msg = f"{where}: {lib().anon_strerror(code).decode()} ({code})"
        if detail:
            msg += f" [{detail}]"
        super().__init__(msg)


_lib = None
_vp, _i32, _i64, _u64, _sz = ctypes.c_void_p, ctypes.c_int32, ctypes.c_int64, ctypes.c_uint64, ctypes.c_size_t

_SIGNATURES = {
    "anon_strerror": (ctypes.c_char_p, [ctypes.c_int]),
    "anon_exported_symbols": (ctypes.POINTER(ctypes.c_char_p), []),
    "anon_ctx_create": (ctypes.c_int, [ctypes.POINTER(_vp), ctypes.c_int, _vp, _sz]),
    "anon_ctx_destroy": (None, [_vp]),
    "anon_ctx_sync": (ctypes.c_int, [_vp]),
    "anon_last_cuda_error": (ctypes.c_char_p, [_vp]),
    "anon_workspace_bytes": (_sz, [ctypes.POINTER(ModelDesc), _i64, _i32]),
    "anon_weights_load": (ctypes.c_int, [_vp, ctypes.POINTER(ModelDesc), _vp, _sz, ctypes.POINTER(_vp)]),
    "anon_weights_free": (None, [_vp]),
    "anon_ner_forward": (ctypes.c_int, [_vp, _vp, _vp, _vp, _i32, _i32, _vp, _vp]),
    "anon_decode_spans": (ctypes.c_int, [_vp, _vp, _vp, _i32, _i32, _vp, _i32, _vp]),
    "anon_decode_spans_static": (ctypes.c_int, [ctypes.c_int, _vp, _vp, _vp, _i32, _i32, _vp, _i32, _vp]),
    "anon_gather_spans": (ctypes.c_int, [_vp, _vp, _vp, _vp, _i32, _vp, _sz, _vp, _vp]),
    "anon_cache_create": (ctypes.c_int, [_vp, _u64, _u64, ctypes.POINTER(_vp)]),
    "anon_cache_destroy": (None, [_vp]),
    "anon_cache_clear": (ctypes.c_int, [_vp]),
    "anon_cache_stats": (ctypes.c_int, [_vp, ctypes.POINTER(_u64), ctypes.POINTER(_u64), ctypes.POINTER(_u64)]),
    "anon_cache_entry": (_i64, [_vp, _u64, _vp, _sz, _vp]),
    "anon_cache_export": (ctypes.c_int, [_vp, _vp, _sz, _vp, _vp, ctypes.POINTER(_u64), ctypes.POINTER(_u64)]),
    "anon_cache_track_use": (ctypes.c_int, [_vp, ctypes.c_int]),
    "anon_cache_evict": (ctypes.c_int, [_vp, _u64, ctypes.POINTER(_u64)]),
    "anon_pseudonymize": (ctypes.c_int, [_vp, _vp, _vp, _vp, _vp, _i64, _vp, _sz, _i32,
                                         ctypes.POINTER(ctypes.c_char_p), _i32, _vp, _sz, _vp, _vp, _vp, _vp]),
    "anon_hmac_spans": (ctypes.c_int, [_vp, _vp, _vp, _i64, _vp, _sz, _vp]),
    "anon_pipeline_host": (ctypes.c_int, [_vp, _vp, _vp, _vp, _vp, _i32, _i32, _vp, _vp, _sz, _vp, _i32, _vp, _sz, _i32,
                                          ctypes.POINTER(ctypes.c_char_p), _i32, _vp, _i32, _vp, _vp, _sz, _vp, _vp]),
    "anon_pipeline_host_text": (ctypes.c_int, [_vp, _vp, _vp, _vp, _vp, _i32, _i32, _vp, _vp, _sz, _vp, _i32, _vp, _sz, _i32,
                                               ctypes.POINTER(ctypes.c_char_p), _i32, _vp, _i32, _vp, _vp, _sz, _vp, _vp,
                                               _vp, _sz, _vp]),
    "anon_ctx_profile": (ctypes.c_int, [_vp, ctypes.c_int]),
    "anon_ctx_profile_read": (ctypes.c_int, [_vp, _vp, _vp, _vp, _vp]),
    "anon_gemm_bf16": (ctypes.c_int, [_vp, _vp, _vp, _vp, _vp, _vp, _i32, _i32, _i32, _i32]),
    "anon_splice_records": (ctypes.c_int, [_vp, _vp, _sz, _vp, _i32, _vp, _i32, _vp, _vp, _vp, _sz, _vp]),
    "anon_attention": (ctypes.c_int, [_vp, _vp, _vp, _vp, _i32, _i32, _i32, _i32, _i32, _vp]),
    "anon_attention_local": (ctypes.c_int, [_vp, _vp, _vp, _vp, _i32, _i32, _i32, _i32, _i32, _i32, _vp]),
    "anon_regex_load": (ctypes.c_int, [_vp, _vp, _sz, ctypes.POINTER(_vp)]),
    "anon_regex_free": (None, [_vp]),
    "anon_regex_scan": (ctypes.c_int, [_vp, _vp, _vp, _sz, _vp, _i32, _vp, _i32, _vp]),
    "anon_merge_spans": (ctypes.c_int, [_vp, _vp, _vp, _i32, _vp, _vp, _i32, _vp, _i32, _vp]),
    "anon_ctx_set_regex": (ctypes.c_int, [_vp, _vp]),
    "anon_gemm_bf16_fold_res": (ctypes.c_int, [_vp, _vp, _vp, _vp, _vp, _vp, _vp, _vp, _vp, ctypes.c_float, _vp, _vp, _vp, _i32, _i32, _i32]),
    "anon_gemm_bf16_fold": (ctypes.c_int, [_vp, _vp, _vp, _vp, _vp, _vp, _i32, ctypes.c_float, _vp, _i32, _i32, _i32]),
    "anon_microbench": (ctypes.c_int, [_vp, _i32, _i32, ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_double)]),
}


def lib():
    """Loads (building if needed) libanonshield.so and declares every prototype of include/anonshield.h."""
    global _lib
    if _lib is None:
        path = _build.build()
        L = ctypes.CDLL(path)
        for name, (res, args) in _SIGNATURES.items():
            fn = getattr(L, name)          # AttributeError here = the library does not export the symbol
            fn.restype = res
            fn.argtypes = args
        _lib = L
    return _lib


def _ptr(t):
    """Device (torch) or host (numpy) buffer -> raw address; None -> NULL."""
    if t is None:
        return None
    if isinstance(t, np.ndarray):
        assert t.flags["C_CONTIGUOUS"]
        return t.ctypes.data
    assert t.is_contiguous()
    return t.data_ptr()


def _names(type_names):
    return (ctypes.c_char_p * len(type_names))(*[t.encode() for t in type_names])


class Context:
    """anon_ctx: one per host thread; enqueues on the given torch stream (default: current stream)."""

    def __init__(self, device=0, workspace_bytes=0, stream=None):
        import torch
        self._h = _vp()
        self.device = device
        if torch.cuda.is_available():
            torch.cuda.set_device(device)
            self.stream = stream if stream is not None else torch.cuda.current_stream(device)
            sp = self.stream.cuda_stream
        else:
            self.stream, sp = None, 0
        rc = lib().anon_ctx_create(ctypes.byref(self._h), device, sp, workspace_bytes)
        if rc:
            raise AnonError(rc, "anon_ctx_create")

    def check(self, rc, where):
        if rc:
            raise AnonError(rc, where, lib().anon_last_cuda_error(self._h).decode() if rc == ERR_CUDA else "")

    def sync(self):
        """anon_ctx_sync: waits for the stream, returns (and clears) the sticky device status."""
        return lib().anon_ctx_sync(self._h)

    def profile(self, enable):
        self.check(lib().anon_ctx_profile(self._h, 1 if enable else 0), "anon_ctx_profile")

    def profile_read(self):
        """{class name: (ms, work, launches)}, total kernel launches since profile() was last called."""
        ms, work = np.zeros(8, np.float64), np.zeros(8, np.float64)
        ln, tot = np.zeros(8, np.int64), np.zeros(1, np.int64)
        self.check(lib().anon_ctx_profile_read(self._h, ms.ctypes.data, work.ctypes.data, ln.ctypes.data, tot.ctypes.data),
                   "anon_ctx_profile_read")
        names = ["gemm_qkv", "attention", "row", "decode", "pseudonymize", "gemm_out", "gemm_ffn1", "gemm_ffn2"]
        return {n: (float(ms[i]), float(work[i]), int(ln[i])) for i, n in enumerate(names)}, int(tot[0])

    def close(self):
        if self._h:
            lib().anon_ctx_destroy(self._h)
            self._h = _vp()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def anon_workspace_bytes(desc, max_tokens, max_seqs):
    d = desc if isinstance(desc, ModelDesc) else ModelDesc.from_dict(desc)
    return lib().anon_workspace_bytes(ctypes.byref(d), max_tokens, max_seqs)


class Weights:
    """anon_weights: device copy of the parameters (fixed blob order of include/anonshield.h)."""

    def __init__(self, ctx, desc, host_fp32_blob):
        self.ctx = ctx
        self.desc = dict(desc)
        d = ModelDesc.from_dict(desc)
        blob = np.ascontiguousarray(host_fp32_blob, np.float32)
        self._h = _vp()
        ctx.check(lib().anon_weights_load(ctx._h, ctypes.byref(d), blob.ctypes.data, blob.size, ctypes.byref(self._h)),
                  "anon_weights_load")

    def close(self):
        if self._h:
            lib().anon_weights_free(self._h)
            self._h = _vp()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


class Cache:
    """anon_cache: the GPU entity cache (open addressing, entity bytes + HMAC digests)."""

    def __init__(self, ctx, max_unique, key_arena_bytes):
        self.ctx = ctx
        self._h = _vp()
        ctx.check(lib().anon_cache_create(ctx._h, max_unique, key_arena_bytes, ctypes.byref(self._h)), "anon_cache_create")

    def clear(self):
        self.ctx.check(lib().anon_cache_clear(self._h), "anon_cache_clear")

    def stats(self):
        a, b, c = _u64(), _u64(), _u64()
        self.ctx.check(lib().anon_cache_stats(self._h, ctypes.byref(a), ctypes.byref(b), ctypes.byref(c)), "anon_cache_stats")
        return {"n_unique": a.value, "n_lookups": b.value, "n_hits": c.value}

    def entry(self, uid):
        dig = np.zeros(32, np.uint8)
        n = lib().anon_cache_entry(self._h, uid, None, 0, dig.ctypes.data)
        if n < 0:
            raise AnonError(int(n), "anon_cache_entry")
        buf = np.zeros(max(int(n), 1), np.uint8)
        lib().anon_cache_entry(self._h, uid, buf.ctypes.data, int(n), dig.ctypes.data)
        return buf[:n].tobytes(), dig.tobytes()

    def track_use(self, enable=True):
        """NEXT-5: stamp every entry with the sequence number of the last anon_pseudonymize call that looked it up."""
        self.ctx.check(lib().anon_cache_track_use(self._h, 1 if enable else 0), "anon_cache_track_use")

    def evict(self, keep):
        """Keep the `keep` most recently used entries (call-granular LRU, reading D21); returns the number evicted."""
        n = _u64()
        self.ctx.check(lib().anon_cache_evict(self._h, keep, ctypes.byref(n)), "anon_cache_evict")
        return n.value

    def export(self):
        """The mapping table in uid order: (entity bytes uint8[], offsets int64[U+1], digests uint8[U,32])."""
        n, nb = _u64(), _u64()
        self.ctx.check(lib().anon_cache_export(self._h, None, 0, None, None, ctypes.byref(n), ctypes.byref(nb)), "anon_cache_export")
        data, off = np.zeros(max(nb.value, 1), np.uint8), np.zeros(n.value + 1, np.int64)
        dig = np.zeros((max(n.value, 1), 32), np.uint8)
        self.ctx.check(lib().anon_cache_export(self._h, data.ctypes.data, data.size, off.ctypes.data, dig.ctypes.data,
                                               ctypes.byref(n), ctypes.byref(nb)), "anon_cache_export")
        return data[:nb.value], off, dig[:n.value]

    def close(self):
        if self._h:
            lib().anon_cache_destroy(self._h)
            self._h = _vp()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


class Regex:
    """anon_regex: a pattern automaton on the device.  `blob` comes from regex_dfa.compile_patterns (NEXT-4)."""

    def __init__(self, ctx, blob):
        self.ctx = ctx
        self._h = _vp()
        b = np.frombuffer(bytes(blob), np.uint8)
        ctx.check(lib().anon_regex_load(ctx._h, b.ctypes.data, b.size, ctypes.byref(self._h)), "anon_regex_load")

    def close(self):
        if self._h:
            lib().anon_regex_free(self._h)
            self._h = _vp()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


# ---- the calls (same names as the C ABI) ---------------------------------------------------------------
def anon_ner_forward(ctx, weights, token_ids, cu_seqlens, logits=None, labels=None):
    B, T = cu_seqlens.numel() - 1, token_ids.numel()
    ctx.check(lib().anon_ner_forward(ctx._h, weights._h, _ptr(token_ids), _ptr(cu_seqlens), B, T, _ptr(logits),
                                     _ptr(labels)), "anon_ner_forward")


def anon_decode_spans(ctx, labels, meta, num_labels, spans, num_spans):
    """labels int32[T], meta int32[T,4], spans int32[cap,4], num_spans int32[1] -- all device tensors."""
    ctx.check(lib().anon_decode_spans(ctx._h, _ptr(labels), _ptr(meta), labels.numel(), num_labels, _ptr(spans),
                                      spans.shape[0], _ptr(num_spans)), "anon_decode_spans")


def anon_decode_spans_static(device, cuda_stream, labels, meta, num_labels, spans, num_spans):
    """anon_decode_spans without a context or any allocation (scratch is a static device array; T <= 1,048,576).  Raises AnonError on anything
    but ANON_OK."""
    rc = lib().anon_decode_spans_static(int(device), ctypes.c_void_p(cuda_stream or 0), _ptr(labels), _ptr(meta), labels.numel(),
                                        num_labels, _ptr(spans), spans.shape[0], _ptr(num_spans))
    if rc != 0:
        raise AnonError(rc, "anon_decode_spans_static")


def anon_gather_spans(ctx, text, record_offsets, spans, S, span_bytes, span_offsets, span_type=None):
    ctx.check(lib().anon_gather_spans(ctx._h, _ptr(text), _ptr(record_offsets), _ptr(spans), S, _ptr(span_bytes),
                                      span_bytes.numel(), _ptr(span_offsets), _ptr(span_type)), "anon_gather_spans")


def anon_pseudonymize(ctx, cache, span_bytes, span_offsets, span_type, key, slug_len, type_names, out_tokens,
                      out_offsets, hit=None, uid=None, digests=None):
    S = span_offsets.numel() - 1
    k = np.frombuffer(bytes(key), np.uint8)
    rc = lib().anon_pseudonymize(ctx._h, cache._h, _ptr(span_bytes), _ptr(span_offsets), _ptr(span_type), S,
                                 k.ctypes.data if k.size else None, k.size, slug_len, _names(type_names),
                                 len(type_names), _ptr(out_tokens), out_tokens.numel(), _ptr(out_offsets), _ptr(hit),
                                 _ptr(uid), _ptr(digests))
    ctx.check(rc, "anon_pseudonymize")


def anon_hmac_spans(ctx, span_bytes, span_offsets, key, digests):
    S = span_offsets.numel() - 1
    k = np.frombuffer(bytes(key), np.uint8)
    ctx.check(lib().anon_hmac_spans(ctx._h, _ptr(span_bytes), _ptr(span_offsets), S, k.ctypes.data if k.size else None,
                                    k.size, _ptr(digests)), "anon_hmac_spans")


def anon_gemm_bf16(ctx, A, W, bias, residual, C, epilogue):
    M, K = A.shape
    N = W.shape[0]
    ctx.check(lib().anon_gemm_bf16(ctx._h, _ptr(A), _ptr(W), _ptr(bias), _ptr(residual), _ptr(C), M, N, K, epilogue),
              "anon_gemm_bf16")


def anon_splice_records(ctx, text, record_offsets, spans, S, out_tokens, out_offsets, new_text, new_record_offsets):
    """Device tensors; rewrites the records with every span replaced by its pseudonym token (NEXT-1)."""
    R = record_offsets.numel() - 1
    ctx.check(lib().anon_splice_records(ctx._h, _ptr(text), text.numel(), _ptr(record_offsets), R, _ptr(spans), S,
                                        _ptr(out_tokens), _ptr(out_offsets), _ptr(new_text), new_text.numel(),
                                        _ptr(new_record_offsets)), "anon_splice_records")


def anon_regex_scan(ctx, regex, text, record_offsets, spans, num_spans):
    """text uint8[n], record_offsets int64[R+1], spans int32[cap,4], num_spans int32[1] -- device tensors (NEXT-4)."""
    R = record_offsets.numel() - 1
    ctx.check(lib().anon_regex_scan(ctx._h, regex._h, _ptr(text), text.numel(), _ptr(record_offsets), R, _ptr(spans),
                                    spans.shape[0], _ptr(num_spans)), "anon_regex_scan")


def anon_merge_spans(ctx, ner_spans, num_ner, regex_spans, num_regex, out_spans, num_out):
    """Span lists int32[n,4] on the device; num_ner / num_regex: device int32[1] tensors or None (= the whole list)."""
    ctx.check(lib().anon_merge_spans(ctx._h, _ptr(ner_spans), _ptr(num_ner), ner_spans.shape[0], _ptr(regex_spans),
                                     _ptr(num_regex), regex_spans.shape[0], _ptr(out_spans), out_spans.shape[0],
                                     _ptr(num_out)), "anon_merge_spans")


def anon_ctx_set_regex(ctx, regex):
    """Attach (or with None detach) a pattern automaton: anon_pipeline_host then merges regex spans into the NER spans."""
    ctx.check(lib().anon_ctx_set_regex(ctx._h, regex._h if regex is not None else None), "anon_ctx_set_regex")
    ctx._regex = regex            # keeps the handle alive while attached


def anon_attention(ctx, qkv, cu_seqlens_dev, cu_seqlens_host, hidden, heads, dtype, out):
    h = np.ascontiguousarray(cu_seqlens_host, np.int32)
    ctx.check(lib().anon_attention(ctx._h, _ptr(qkv), _ptr(cu_seqlens_dev), h.ctypes.data, h.size - 1, qkv.shape[0],
                                   hidden, heads, dtype, _ptr(out)), "anon_attention")


def anon_attention_local(ctx, qkv, cu_seqlens_dev, cu_seqlens_host, hidden, heads, dtype, window, out):
    h = np.ascontiguousarray(cu_seqlens_host, np.int32)
    ctx.check(lib().anon_attention_local(ctx._h, _ptr(qkv), _ptr(cu_seqlens_dev), h.ctypes.data, h.size - 1, qkv.shape[0],
                                         hidden, heads, dtype, window, _ptr(out)), "anon_attention_local")


def anon_pipeline_host(ctx, weights, cache, token_ids, cu_seqlens, meta, text, record_offsets, key, slug_len,
                       type_names, span_capacity, out_capacity, want_hit=True, bufs=None, want_text=False):
    """Whole hot path on HOST numpy buffers (pinned or pageable).  Returns dict(spans, out_tokens, out_offsets, hit);
    with want_text=True (anon_pipeline_host_text) also new_text and new_record_offsets, the rewritten records."""
    T, B, R = token_ids.size, cu_seqlens.size - 1, record_offsets.size - 1
    if bufs is None:
        bufs = dict(spans=np.zeros((span_capacity, 4), np.int32), out=np.zeros(out_capacity, np.uint8),
                    off=np.zeros(span_capacity + 1, np.int64), hit=np.zeros(span_capacity, np.uint8))
    n = _i32(0)
    k = np.frombuffer(bytes(key), np.uint8)
    args = [ctx._h, weights._h, cache._h, _ptr(token_ids), _ptr(cu_seqlens), B, T, _ptr(meta),
            _ptr(text), text.size, _ptr(record_offsets), R, k.ctypes.data if k.size else None, k.size,
            slug_len, _names(type_names), len(type_names), _ptr(bufs["spans"]), span_capacity,
            ctypes.byref(n), _ptr(bufs["out"]), out_capacity, _ptr(bufs["off"]),
            _ptr(bufs["hit"]) if want_hit else None]
    if want_text:
        if "new_text" not in bufs:
            bufs["new_text"] = np.zeros(text.size + out_capacity, np.uint8)
            bufs["new_ro"] = np.zeros(R + 1, np.int64)
        rc = lib().anon_pipeline_host_text(*args, _ptr(bufs["new_text"]), bufs["new_text"].size, _ptr(bufs["new_ro"]))
        ctx.check(rc, "anon_pipeline_host_text")
    else:
        ctx.check(lib().anon_pipeline_host(*args), "anon_pipeline_host")
    S = n.value
    off = bufs["off"][:S + 1]
    res = {"spans": bufs["spans"][:S], "out_tokens": bufs["out"][:off[S]], "out_offsets": off, "hit": bufs["hit"][:S]}
    if want_text:
        ro = bufs["new_ro"][:R + 1]
        res["new_record_offsets"] = ro
        res["new_text"] = bufs["new_text"][:ro[R]]
    return res


def anon_microbench(ctx, mode, iters=2048):
    """Measured issue rate of the integer-ALU (modes 0-3) or MUFU ex2 (mode 4) pipe: (thread-ops per second, kernel ms)."""
    ops, ms = ctypes.c_double(0.0), ctypes.c_double(0.0)
    ctx.check(lib().anon_microbench(ctx._h, mode, iters, ctypes.byref(ops), ctypes.byref(ms)), "anon_microbench")
    return ops.value, ms.value


def anon_gemm_bf16_fold_res(ctx, A, W, bias, res, res_part, res_stats, gamma, beta, eps, C, Cb, part_out):
    """Producer of the LayerNorm fold: C = A W^T + bias + LN(res) (FP32), Cb = bf16(C), part_out = partial row statistics."""
    M, K = A.shape
    N = W.shape[0]
    ctx.check(lib().anon_gemm_bf16_fold_res(ctx._h, _ptr(A), _ptr(W), _ptr(bias), _ptr(res), _ptr(res_part), _ptr(res_stats), _ptr(gamma),
                                            _ptr(beta), eps, _ptr(C), _ptr(Cb), _ptr(part_out), M, N, K), "anon_gemm_bf16_fold_res")


def anon_gemm_bf16_fold(ctx, A_raw, Wf, c, s, part, stat_cols, eps, C):
    """Consumer of the LayerNorm fold: C = rstd * (A_raw Wf^T - mean * s) + c (BF16)."""
    M, K = A_raw.shape
    N = Wf.shape[0]
    ctx.check(lib().anon_gemm_bf16_fold(ctx._h, _ptr(A_raw), _ptr(Wf), _ptr(c), _ptr(s), _ptr(part), stat_cols, eps, _ptr(C), M, N, K),
              "anon_gemm_bf16_fold")
