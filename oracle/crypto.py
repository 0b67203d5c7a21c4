"""TEST INFRASTRUCTURE -- ctypes front of oracle/anon_oracle.c (plain C, single thread).

Follows PAPER.md L43-L44, L50, L52 and SURVEY.md §8(c) O4; see the C file's header.
"""
import ctypes
import hashlib
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "anon_oracle.c")
_SO = os.path.join(_HERE, "liboracle.so")
_STAMP = _SO + ".stamp"
_CFLAGS = ["-O2", "-std=c11", "-shared", "-fPIC", "-Wall"]


def _src_digest():
    h = hashlib.sha256()
    with open(_SRC, "rb") as f:
        h.update(f.read())
    h.update(" ".join(_CFLAGS).encode())
    return h.hexdigest()


def build(force=False):
    """Compile anon_oracle.c with gcc (building the checker is not using it)."""
    want = _src_digest()
    if not force and os.path.exists(_SO) and os.path.exists(_STAMP):
        with open(_STAMP) as f:
            if f.read().strip() == want:
                return _SO
    subprocess.check_call(["gcc", *_CFLAGS, "-o", _SO, _SRC])
    with open(_STAMP, "w") as f:
        f.write(want)
    return _SO


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = ctypes.CDLL(build())
        u8p, i64p, vp = ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p
        L.oracle_sha256.argtypes = [u8p, ctypes.c_uint64, u8p]
        L.oracle_hmac_sha256.argtypes = [u8p, ctypes.c_uint64, u8p, ctypes.c_uint64, u8p]
        L.oracle_hmac_batch.argtypes = [u8p, ctypes.c_uint64, u8p, i64p, ctypes.c_int64, u8p]
        L.oracle_sha256_constants.argtypes = [vp, vp]
        L.oracle_cache_create.restype = ctypes.c_void_p
        L.oracle_cache_create.argtypes = [ctypes.c_uint64]
        L.oracle_cache_destroy.argtypes = [ctypes.c_void_p]
        L.oracle_cache_stats.argtypes = [ctypes.c_void_p, vp, vp, vp]
        L.oracle_cache_entry.restype = ctypes.c_int64
        L.oracle_cache_entry.argtypes = [ctypes.c_void_p, ctypes.c_int64, u8p, ctypes.c_uint64, u8p]
        L.oracle_pseudonymize.restype = ctypes.c_int
        L.oracle_pseudonymize.argtypes = [
            ctypes.c_void_p, u8p, i64p, u8p, ctypes.c_int64, u8p, ctypes.c_uint64, ctypes.c_int32,
            ctypes.POINTER(ctypes.c_char_p), ctypes.c_int32, u8p, ctypes.c_uint64, i64p, u8p, i64p, u8p]
        _lib = L
    return _lib


def _buf(b):
    a = np.frombuffer(bytes(b), dtype=np.uint8) if not isinstance(b, np.ndarray) else b
    return a, (a.ctypes.data if a.size else None)


def sha256(msg):
    a, p = _buf(msg)
    out = np.zeros(32, np.uint8)
    lib().oracle_sha256(p, a.size, out.ctypes.data)
    return out.tobytes()


def hmac_sha256(key, msg):
    k, kp = _buf(key)
    a, p = _buf(msg)
    out = np.zeros(32, np.uint8)
    lib().oracle_hmac_sha256(kp, k.size, p, a.size, out.ctypes.data)
    return out.tobytes()


def sha256_constants():
    k = np.zeros(64, np.uint32)
    h = np.zeros(8, np.uint32)
    lib().oracle_sha256_constants(k.ctypes.data, h.ctypes.data)
    return k, h


def hmac_batch(key, span_bytes, span_offsets):
    k, kp = _buf(key)
    sb = np.ascontiguousarray(span_bytes, np.uint8)
    so = np.ascontiguousarray(span_offsets, np.int64)
    n = so.size - 1
    out = np.zeros((n, 32), np.uint8)
    lib().oracle_hmac_batch(kp, k.size, sb.ctypes.data, so.ctypes.data, n, out.ctypes.data)
    return out


class Cache:
    """The map M of SURVEY §8(c) O4 (unbounded, no eviction; bound to its first key)."""

    def __init__(self, nbuckets=1 << 20):
        self._h = lib().oracle_cache_create(nbuckets)

    def close(self):
        if self._h:
            lib().oracle_cache_destroy(self._h)
            self._h = None

    __del__ = close

    def stats(self):
        a, b, c = (ctypes.c_int64(), ctypes.c_int64(), ctypes.c_int64())
        lib().oracle_cache_stats(self._h, ctypes.addressof(a), ctypes.addressof(b), ctypes.addressof(c))
        return {"n_unique": a.value, "n_lookups": b.value, "n_hits": c.value}

    def entry(self, uid):
        d = np.zeros(32, np.uint8)
        n = lib().oracle_cache_entry(self._h, uid, None, 0, d.ctypes.data)
        if n < 0:
            raise KeyError(uid)
        b = np.zeros(max(n, 1), np.uint8)
        lib().oracle_cache_entry(self._h, uid, b.ctypes.data, n, d.ctypes.data)
        return b[:n].tobytes(), d.tobytes()

    def pseudonymize(self, span_bytes, span_offsets, span_type, key, slug_len, type_names):
        """Returns dict(out_tokens, out_offsets, hit, uid, digests) as numpy arrays."""
        sb = np.ascontiguousarray(span_bytes, np.uint8)
        so = np.ascontiguousarray(span_offsets, np.int64)
        S = so.size - 1
        st = None if span_type is None else np.ascontiguousarray(span_type, np.uint8)
        k, kp = _buf(key)
        names = (ctypes.c_char_p * len(type_names))(*[t.encode() for t in type_names])
        cap = int(S) * (3 + max(len(t) for t in type_names) + slug_len)
        out = np.zeros(max(cap, 1), np.uint8)
        off = np.zeros(S + 1, np.int64)
        hit = np.zeros(max(S, 1), np.uint8)
        uid = np.zeros(max(S, 1), np.int64)
        dig = np.zeros((max(S, 1), 32), np.uint8)
        rc = lib().oracle_pseudonymize(
            self._h, sb.ctypes.data if sb.size else None, so.ctypes.data,
            None if st is None else st.ctypes.data, S, kp, k.size, slug_len, names, len(type_names),
            out.ctypes.data, cap, off.ctypes.data, hit.ctypes.data, uid.ctypes.data, dig.ctypes.data)
        if rc == -1:
            raise KeyError("cache is bound to another key")
        if rc != 0:
            raise ValueError(f"oracle_pseudonymize rc={rc}")
        return {"out_tokens": out[: off[S]], "out_offsets": off, "hit": hit[:S], "uid": uid[:S],
                "digests": dig[:S]}
