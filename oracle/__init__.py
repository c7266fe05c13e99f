"""ORACLE — TEST INFRASTRUCTURE, NOT PRODUCT CODE.

ctypes wrapper around the plain-C oracle (``oracle/*.c``): the CPU encoder and the two CPU
decoders of the format in ``/FORMAT.md``. Only ``tests/``, ``__graft_entry__.smoke()`` and
``bench.py`` (input preparation, ``cpu_baseline`` and ``--impl reference``) may import this
package. It never imports ``paper_2606_24531_b200`` and shares no code with the CUDA path.
See ``aceapex_oracle.h`` for the citations of each function.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
import threading

import numpy as np

_DIR = os.path.dirname(os.path.abspath(__file__))
# Block size: 16 KiB (block_log2 14). ACEAPEX_BLOCK_LOG2=12..15 selects a variant of the oracle compiled
# with -DORA_BLOG for the block-size sweep (`bench.py --sweep`).
BLOG = int(os.environ.get("ACEAPEX_BLOCK_LOG2", "14"))
if not 12 <= BLOG <= 15:
    raise ValueError("ACEAPEX_BLOCK_LOG2 must be 12..15")
_SO = os.path.join(_DIR, "libaceapex_oracle.so" if BLOG == 14 else f"libaceapex_oracle_b{BLOG}.so")
_SRC = ["rans.c", "decoder.c", "encoder.c"]
_HDR = ["aceapex_oracle.h", "container.h"]
_lock = threading.Lock()
_lib = None

B = 1 << BLOG
MAX_SEQ = B // 4
LIT, LEN, OFF = 0, 1, 2


class OracleError(RuntimeError):
    def __init__(self, code: int, what: str):
        super().__init__(f"oracle: {what}: code {code}")
        self.code = code


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (plain C11, OpenMP only for the encoder's block loop)."""
    srcs = [os.path.join(_DIR, s) for s in _SRC]
    deps = srcs + [os.path.join(_DIR, h) for h in _HDR]
    if not force and os.path.exists(_SO) and all(os.path.getmtime(_SO) >= os.path.getmtime(d) for d in deps):
        return _SO
    tmp = _SO + f".tmp{os.getpid()}"
    cmd = ["gcc", "-std=c11", "-O2", "-g", "-fopenmp", "-fPIC", "-shared", "-Wall", "-Wextra", f"-DORA_BLOG={BLOG}", "-o", tmp] + srcs
    subprocess.run(cmd, check=True, cwd=_DIR)
    os.replace(tmp, _SO)
    return _SO


class EncParams(C.Structure):
    _fields_ = [(n, C.c_uint32) for n in
                ("min_match", "chain_depth", "max_depth", "window", "max_level", "offset_width", "threads", "batch",
                 "raw_slack_pct", "max_fanout", "long_hash", "long_chain", "max_seq")]


class EncStats(C.Structure):
    _fields_ = [("n_seq", C.c_uint64), ("n_lit", C.c_uint64), ("match_bytes", C.c_uint64),
                ("intra_match_bytes", C.c_uint64), ("n_extras", C.c_uint64),
                ("n_sym", C.c_uint64 * 3), ("n_words", C.c_uint64 * 3), ("table_bytes", C.c_uint64),
                ("max_depth_seen", C.c_uint32), ("max_level_seen", C.c_uint32), ("n_raw", C.c_uint64 * 3),
                ("n_const", C.c_uint64 * 3)]


class Info(C.Structure):
    _fields_ = [("total_len", C.c_uint64), ("n_blocks", C.c_uint64), ("payload_off", C.c_uint64),
                ("container_bytes", C.c_uint64), ("offset_width", C.c_uint32), ("max_depth", C.c_uint32),
                ("window", C.c_uint32), ("max_level", C.c_uint32), ("min_match_policy", C.c_uint32),
                ("max_fanout", C.c_uint32)]


class BlockHdr(C.Structure):
    _fields_ = [("n_seq", C.c_uint32), ("n_lit", C.c_uint32), ("n_extras", C.c_uint32),
                ("off_nbytes", C.c_uint32), ("n_sym", C.c_uint32 * 3), ("n_words", C.c_uint32 * 3)]


class ValidateReport(C.Structure):
    _fields_ = [("n_seq", C.c_uint64), ("n_matches_cross", C.c_uint64), ("n_matches_intra", C.c_uint64),
                ("n_matches_spanning", C.c_uint64), ("max_depth_seen", C.c_uint32),
                ("max_level_seen", C.c_uint32), ("min_match_seen", C.c_uint32),
                ("max_src_blocks_per_block", C.c_uint32), ("mean_src_blocks_per_block", C.c_double)]


def lib():
    global _lib
    with _lock:
        if _lib is None:
            L = C.CDLL(build())
            vp, sz, u8p = C.c_void_p, C.c_size_t, C.c_void_p
            L.ora_quantise.argtypes = [vp, vp]; L.ora_quantise.restype = None
            L.ora_rans_encode.argtypes = [u8p, sz, vp, C.c_uint32, vp, vp, C.POINTER(sz)]
            L.ora_rans_decode.argtypes = [vp, C.c_uint32, vp, sz, vp, u8p, sz]
            L.ora_fnv1a64.argtypes = [vp, sz]; L.ora_fnv1a64.restype = C.c_uint64
            L.ora_enc_params_default.argtypes = [C.POINTER(EncParams)]; L.ora_enc_params_default.restype = None
            L.ora_encode_bound.argtypes = [sz]; L.ora_encode_bound.restype = sz
            L.ora_encode.argtypes = [u8p, sz, C.POINTER(EncParams), u8p, sz, C.POINTER(sz), C.POINTER(EncStats)]
            L.ora_info_get.argtypes = [u8p, sz, C.POINTER(Info)]
            L.ora_decode_streams.argtypes = [u8p, sz, C.c_uint64, C.POINTER(BlockHdr), vp, vp, vp, vp, vp]
            L.ora_decode_tokens.argtypes = [u8p, sz, C.c_uint64, C.POINTER(C.c_uint32), vp, vp, vp, vp]
            L.ora_decode_all.argtypes = [u8p, sz, u8p, sz]
            L.ora_decode_all_mt.argtypes = [u8p, sz, u8p, sz, C.c_uint32]
            L.ora_iso_open.argtypes = [u8p, sz, C.POINTER(vp)]
            L.ora_iso_decode.argtypes = [vp, C.c_uint64, u8p, sz, C.POINTER(C.c_uint32), C.POINTER(C.c_uint32)]
            L.ora_iso_close.argtypes = [vp]; L.ora_iso_close.restype = None
            L.ora_validate.argtypes = [u8p, sz, C.POINTER(ValidateReport)]
            L.ora_strerror.argtypes = [C.c_int]; L.ora_strerror.restype = C.c_char_p
            L.ora_block_log2.restype = C.c_int
            if L.ora_block_log2() != BLOG:
                raise RuntimeError(f"{_SO}: compiled for block_log2 {L.ora_block_log2()}, wanted {BLOG}")
            _lib = L
    return _lib


def _ptr(a: np.ndarray):
    return a.ctypes.data_as(C.c_void_p)


def _bytes_arr(data) -> np.ndarray:
    a = np.frombuffer(data, dtype=np.uint8) if isinstance(data, (bytes, bytearray, memoryview)) else np.asarray(data)
    if a.dtype != np.uint8:
        raise TypeError("expected bytes / uint8 array")
    return np.ascontiguousarray(a)


def _check(rc: int, what: str):
    if rc != 0:
        raise OracleError(rc, f"{what}: {lib().ora_strerror(rc).decode()}")


# ---------------------------------------------------------------- entropy layer

def quantise(count) -> np.ndarray:
    cnt = np.ascontiguousarray(np.asarray(count, dtype=np.uint32))
    assert cnt.shape == (256,)
    freq = np.zeros(256, dtype=np.uint16)
    lib().ora_quantise(_ptr(cnt), _ptr(freq))
    return freq


def rans_encode(sym, freq, lanes: int = 32):
    s = _bytes_arr(sym)
    f = np.ascontiguousarray(np.asarray(freq, dtype=np.uint16))
    states = np.zeros(lanes, dtype=np.uint32)
    words = np.zeros(max(1, s.size), dtype=np.uint16)
    nw = C.c_size_t(0)
    _check(lib().ora_rans_encode(_ptr(s), s.size, _ptr(f), lanes, _ptr(states), _ptr(words), C.byref(nw)), "rans_encode")
    return states, words[: nw.value].copy()


def rans_decode(states, words, freq, n: int, lanes: int = 32) -> np.ndarray:
    st = np.ascontiguousarray(np.asarray(states, dtype=np.uint32))
    w = np.ascontiguousarray(np.asarray(words, dtype=np.uint16))
    f = np.ascontiguousarray(np.asarray(freq, dtype=np.uint16))
    out = np.zeros(max(1, n), dtype=np.uint8)
    _check(lib().ora_rans_decode(_ptr(st), lanes, _ptr(w), w.size, _ptr(f), _ptr(out), n), "rans_decode")
    return out[:n]


def fnv1a64(data) -> int:
    a = _bytes_arr(data)
    return int(lib().ora_fnv1a64(_ptr(a), a.size))


# ---------------------------------------------------------------- codec

def enc_params(**kw) -> EncParams:
    p = EncParams()
    lib().ora_enc_params_default(C.byref(p))
    for k, v in kw.items():
        if not hasattr(p, k):
            raise TypeError(f"unknown encoder parameter {k}")
        setattr(p, k, int(v))
    return p


def encode(data, return_stats: bool = False, **params):
    """Oracle encoder. Returns the container as a uint8 array (and EncStats)."""
    a = _bytes_arr(data)
    p = enc_params(**params)
    cap = lib().ora_encode_bound(a.size)
    out = np.empty(cap, dtype=np.uint8)
    n = C.c_size_t(0)
    st = EncStats()
    _check(lib().ora_encode(_ptr(a), a.size, C.byref(p), _ptr(out), cap, C.byref(n), C.byref(st)), "encode")
    c = out[: n.value].copy()
    return (c, st) if return_stats else c


def info(container) -> Info:
    c = _bytes_arr(container)
    i = Info()
    _check(lib().ora_info_get(_ptr(c), c.size, C.byref(i)), "info")
    return i


def decode_all(container) -> np.ndarray:
    """Decoder #1 (sequential)."""
    c = _bytes_arr(container)
    i = info(c)
    out = np.full(max(1, i.total_len), 0xA5, dtype=np.uint8)
    _check(lib().ora_decode_all(_ptr(c), c.size, _ptr(out), i.total_len), "decode_all")
    return out[: i.total_len]


def decode_all_mt(container, threads: int) -> np.ndarray:
    """Decoder #1 with the entropy stage on `threads` host threads, the match stage in block order."""
    c = _bytes_arr(container)
    i = info(c)
    out = np.full(max(1, i.total_len), 0xA5, dtype=np.uint8)
    _check(lib().ora_decode_all_mt(_ptr(c), c.size, _ptr(out), i.total_len, threads), "decode_all_mt")
    return out[: i.total_len]


def decode_streams(container, block: int):
    """Entropy-decode one block: (hdr, lit, len, off, extras, tags)."""
    c = _bytes_arr(container)
    h = BlockHdr()
    lit = np.zeros(B, np.uint8); ln = np.zeros(2 * MAX_SEQ, np.uint8); off = np.zeros(8 * MAX_SEQ, np.uint8)
    ex = np.zeros(2 * MAX_SEQ, np.uint16); tags = np.zeros(MAX_SEQ, np.uint8)
    _check(lib().ora_decode_streams(_ptr(c), c.size, block, C.byref(h), _ptr(lit), _ptr(ln), _ptr(off), _ptr(ex), _ptr(tags)),
           "decode_streams")
    return (h, lit[: h.n_sym[LIT]].copy(), ln[: h.n_sym[LEN]].copy(), off[: h.n_sym[OFF]].copy(),
            ex[: h.n_extras].copy(), tags[: h.n_seq].copy())


def decode_tokens(container, block: int):
    """Parsed tokens of one block: (lit_len, match_len, src, tags)."""
    c = _bytes_arr(container)
    n = C.c_uint32(0)
    ll = np.zeros(MAX_SEQ, np.uint32); ml = np.zeros(MAX_SEQ, np.uint32); src = np.zeros(MAX_SEQ, np.uint64)
    tags = np.zeros(MAX_SEQ, np.uint8)
    _check(lib().ora_decode_tokens(_ptr(c), c.size, block, C.byref(n), _ptr(ll), _ptr(ml), _ptr(src), _ptr(tags)),
           "decode_tokens")
    k = n.value
    return ll[:k].copy(), ml[:k].copy(), src[:k].copy(), tags[:k].copy()


class Isolated:
    """Decoder #2 (per-byte origin chase), memoising parsed blocks."""

    def __init__(self, container):
        self._c = _bytes_arr(container)  # keep alive
        self._h = C.c_void_p()
        _check(lib().ora_iso_open(_ptr(self._c), self._c.size, C.byref(self._h)), "iso_open")

    def decode(self, block: int, with_hops: bool = False):
        dst = np.full(B, 0x5A, dtype=np.uint8)
        n = C.c_uint32(0); hops = C.c_uint32(0)
        _check(lib().ora_iso_decode(self._h, block, _ptr(dst), B, C.byref(n), C.byref(hops)), "iso_decode")
        return (dst[: n.value].copy(), hops.value) if with_hops else dst[: n.value].copy()

    def close(self):
        if self._h:
            lib().ora_iso_close(self._h)
            self._h = C.c_void_p()

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def validate(container) -> ValidateReport:
    c = _bytes_arr(container)
    rep = ValidateReport()
    _check(lib().ora_validate(_ptr(c), c.size, C.byref(rep)), "validate")
    return rep
