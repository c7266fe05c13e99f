"""Thin ctypes binding over the C-ABI library ``libaceapex.so`` (``include/aceapex.h``).

Argument marshalling only: every step of the decode runs in the CUDA kernels of ``csrc/``.
PyTorch is used for device memory and streams, nothing else. There is no CPU fallback: if the
library is not built, or no CUDA device is present, the calls raise.
"""
from __future__ import annotations

import ctypes as C
import os
import threading

import numpy as np

from . import build as _build

# Block size: 16 KiB unless the library variant loaded through ACEAPEX_LIB was built for another one (block-size sweep,
# `bench.py --sweep`), in which case ACEAPEX_BLOCK_LOG2 names it; aceapex_open rejects a container of any other size.
BLOG = int(os.environ.get("ACEAPEX_BLOCK_LOG2", "14"))
B = 1 << BLOG
PACKED, ABSOLUTE = 0, 1

ERRORS = {0: "OK", -1: "E_ARG", -2: "E_FORMAT", -3: "E_CAPACITY", -4: "E_CORRUPT", -5: "E_RANGE",
          -6: "E_NOMEM", -7: "E_CUDA", -8: "E_STATE"}
E_ARG, E_FORMAT, E_CAPACITY, E_CORRUPT, E_RANGE, E_NOMEM, E_CUDA, E_STATE = -1, -2, -3, -4, -5, -6, -7, -8

# every symbol include/aceapex.h declares
SYMBOLS = ["aceapex_version", "aceapex_open", "aceapex_info_get", "aceapex_scratch_bytes", "aceapex_set_scratch",
           "aceapex_decode_all", "aceapex_decode_range", "aceapex_decode_blocks", "aceapex_seek", "aceapex_device_status",
           "aceapex_launch_count", "aceapex_decode_streams", "aceapex_profile_enable", "aceapex_profile_read",
           "aceapex_kernel_name", "aceapex_strerror", "aceapex_close", "aceapex_decode_all_static"]
N_KERNELS = 16


class AceapexError(RuntimeError):
    def __init__(self, code: int, what: str):
        super().__init__(f"{what}: {ERRORS.get(code, code)} ({lib().aceapex_strerror(code).decode()})")
        self.code = code


class Info(C.Structure):
    _fields_ = [("total_len", C.c_uint64), ("n_blocks", C.c_uint64), ("container_bytes", C.c_uint64),
                ("block_size", C.c_uint32), ("offset_width", C.c_uint32), ("max_depth", C.c_uint32),
                ("window", C.c_uint32), ("max_level", C.c_uint32), ("max_n_seq", C.c_uint32)]


_lock = threading.Lock()
_lib = None


def lib_path() -> str:
    return _build.SO


def lib():
    """Load libaceapex.so (building it with nvcc if it is missing or stale). Fails loudly."""
    global _lib
    with _lock:
        if _lib is None:
            # ACEAPEX_LIB: a variant built by build.build_variant (granularity sweeps); otherwise the in-tree library
            path = os.environ.get("ACEAPEX_LIB") or _build.build()
            if not os.path.exists(path):
                raise RuntimeError(f"{path}: CUDA library not found (there is no CPU fallback)")
            L = C.CDLL(path)
            vp, sz, u64, u32 = C.c_void_p, C.c_size_t, C.c_uint64, C.c_uint32
            L.aceapex_version.restype = C.c_int
            L.aceapex_open.argtypes = [vp, sz, vp, C.POINTER(vp)]
            L.aceapex_info_get.argtypes = [vp, C.POINTER(Info)]
            L.aceapex_scratch_bytes.argtypes = [vp, sz, sz]; L.aceapex_scratch_bytes.restype = sz
            L.aceapex_set_scratch.argtypes = [vp, vp, sz, sz, sz, vp]
            L.aceapex_decode_all.argtypes = [vp, vp, sz, vp]
            L.aceapex_decode_range.argtypes = [vp, u64, u64, vp, sz, vp]
            L.aceapex_decode_blocks.argtypes = [vp, vp, sz, vp, sz, u32, vp]
            L.aceapex_seek.argtypes = [vp, u64, vp, sz, C.POINTER(u64), C.POINTER(u32), vp]
            L.aceapex_device_status.argtypes = [vp, vp, C.POINTER(u64), C.c_int]
            L.aceapex_launch_count.argtypes = [vp]; L.aceapex_launch_count.restype = u64
            L.aceapex_decode_streams.argtypes = [vp, u64, sz, vp, vp, vp, vp]
            L.aceapex_profile_enable.argtypes = [vp, C.c_int]
            L.aceapex_profile_read.argtypes = [vp, vp, vp]
            L.aceapex_kernel_name.argtypes = [C.c_int]; L.aceapex_kernel_name.restype = C.c_char_p
            L.aceapex_strerror.argtypes = [C.c_int]; L.aceapex_strerror.restype = C.c_char_p
            L.aceapex_close.argtypes = [vp]; L.aceapex_close.restype = None
            L.aceapex_decode_all_static.argtypes = [vp, sz, vp, u32, vp, sz, vp, vp]
            _lib = L
    return _lib


def _check(rc: int, what: str):
    if rc != 0:
        raise AceapexError(rc, what)


def _stream_ptr(stream) -> int:
    import torch
    s = torch.cuda.current_stream() if stream is None else stream
    return int(s.cuda_stream)


class Decoder:
    """One opened container resident in device memory (``aceapex_open`` .. ``aceapex_close``)."""

    def __init__(self, container, n_slots: int | None = None, n_targets: int = 256, device="cuda:0"):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("paper_2606_24531_b200 needs a CUDA device (sm_100a); there is no CPU fallback")
        self._torch = torch
        self.device = torch.device(device)
        L = lib()
        if isinstance(container, torch.Tensor):
            t = container.to(self.device, dtype=torch.uint8).contiguous()
        else:
            host = np.ascontiguousarray(np.frombuffer(container, dtype=np.uint8) if isinstance(container, (bytes, bytearray, memoryview))
                                        else np.asarray(container, dtype=np.uint8))
            t = torch.from_numpy(host).to(self.device)
        if t.data_ptr() % 16:
            raise ValueError("container tensor must be 16-byte aligned")
        self.container = t
        self._ctx = C.c_void_p()
        with torch.cuda.device(self.device):
            _check(L.aceapex_open(t.data_ptr(), t.numel(), None, C.byref(self._ctx)), "aceapex_open")
        self.info = Info()
        _check(L.aceapex_info_get(self._ctx, C.byref(self.info)), "aceapex_info_get")
        self.scratch = None
        self.set_scratch(n_slots if n_slots is not None else max(1, min(int(self.info.n_blocks), 65536)), n_targets)

    # -- aceapex_scratch_bytes / aceapex_set_scratch
    def set_scratch(self, n_slots: int, n_targets: int, stream=None):
        torch = self._torch
        L = lib()
        need = L.aceapex_scratch_bytes(self._ctx, n_slots, n_targets)
        self.scratch = torch.empty(need + 256, dtype=torch.uint8, device=self.device)
        off = (-self.scratch.data_ptr()) % 256
        self._scratch_view = self.scratch[off:off + need]
        self.n_slots, self.n_targets = n_slots, n_targets
        with torch.cuda.device(self.device):
            _check(L.aceapex_set_scratch(self._ctx, self._scratch_view.data_ptr(), need, n_slots, n_targets,
                                         _stream_ptr(stream)), "aceapex_set_scratch")

    # -- aceapex_decode_all
    def decode_all(self, out=None, stream=None):
        torch = self._torch
        if out is None:
            out = torch.empty(max(1, int(self.info.total_len)), dtype=torch.uint8, device=self.device)
        with torch.cuda.device(self.device):
            _check(lib().aceapex_decode_all(self._ctx, out.data_ptr(), out.numel(), _stream_ptr(stream)), "aceapex_decode_all")
        return out

    # -- aceapex_decode_range
    def decode_range(self, first: int, count: int, out=None, stream=None):
        """Blocks [first, first+count) into a range-sized buffer (block first+i at out[i*16384:])."""
        torch = self._torch
        if out is None:
            out = torch.empty(max(1, count * B), dtype=torch.uint8, device=self.device)
        with torch.cuda.device(self.device):
            _check(lib().aceapex_decode_range(self._ctx, int(first), int(count), out.data_ptr(), out.numel(),
                                              _stream_ptr(stream)), "aceapex_decode_range")
        return out

    # -- aceapex_decode_blocks
    def decode_blocks(self, ids, out=None, flags: int = PACKED, stream=None):
        torch = self._torch
        ids = np.ascontiguousarray(np.asarray(ids, dtype=np.uint64))
        if out is None:
            n = len(ids) * B if flags == PACKED else int(self.info.n_blocks) * B
            out = torch.empty(max(1, n), dtype=torch.uint8, device=self.device)
        with torch.cuda.device(self.device):
            _check(lib().aceapex_decode_blocks(self._ctx, ids.ctypes.data_as(C.c_void_p), len(ids), out.data_ptr(),
                                               out.numel(), flags, _stream_ptr(stream)), "aceapex_decode_blocks")
        return out

    # -- aceapex_seek
    def seek(self, coord: int, out=None, stream=None):
        """Returns (tensor holding the enclosing block, block_start, block_len)."""
        torch = self._torch
        if out is None:
            out = torch.empty(B, dtype=torch.uint8, device=self.device)
        start, length = C.c_uint64(0), C.c_uint32(0)
        with torch.cuda.device(self.device):
            _check(lib().aceapex_seek(self._ctx, int(coord), out.data_ptr(), out.numel(), C.byref(start), C.byref(length),
                                      _stream_ptr(stream)), "aceapex_seek")
        return out, start.value, length.value

    # -- aceapex_decode_streams (test / profiling hook)
    def decode_streams(self, first: int, count: int, stream=None):
        torch = self._torch
        lit = torch.zeros(count * B, dtype=torch.uint8, device=self.device)
        ln = torch.zeros(count * (B // 2), dtype=torch.uint8, device=self.device)
        off = torch.zeros(count * (2 * B), dtype=torch.uint8, device=self.device)
        with torch.cuda.device(self.device):
            _check(lib().aceapex_decode_streams(self._ctx, first, count, lit.data_ptr(), ln.data_ptr(), off.data_ptr(),
                                                _stream_ptr(stream)), "aceapex_decode_streams")
        return lit, ln, off

    # -- aceapex_device_status
    def device_status(self, clear: bool = False, stream=None):
        """Synchronises; returns (code, first_bad_block)."""
        bad = C.c_uint64(0)
        with self._torch.cuda.device(self.device):
            rc = lib().aceapex_device_status(self._ctx, _stream_ptr(stream), C.byref(bad), 1 if clear else 0)
        return rc, bad.value

    def check(self, stream=None):
        rc, bad = self.device_status(stream=stream)
        if rc != 0:
            raise AceapexError(rc, f"device status (first bad block {bad})")

    # -- aceapex_profile_enable / aceapex_profile_read
    def profile_enable(self, on: bool = True):
        _check(lib().aceapex_profile_enable(self._ctx, 1 if on else 0), "aceapex_profile_enable")

    def profile_read(self) -> dict:
        """{kernel name: (launches, summed device ms)} since the last read; synchronises."""
        n = (C.c_uint64 * N_KERNELS)()
        ms = (C.c_double * N_KERNELS)()
        _check(lib().aceapex_profile_read(self._ctx, n, ms), "aceapex_profile_read")
        out = {}
        for i in range(N_KERNELS):
            name = lib().aceapex_kernel_name(i)
            if name and n[i]:
                out[name.decode()] = (int(n[i]), float(ms[i]))
        return out

    @property
    def launch_count(self) -> int:
        return int(lib().aceapex_launch_count(self._ctx))

    def close(self):
        if getattr(self, "_ctx", None) and self._ctx.value:
            lib().aceapex_close(self._ctx)
            self._ctx = C.c_void_p()

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


STATIC_SCRATCH_BYTES = 8 << 20
STATIC_MAX_BLOCKS = 4096


def decode_all_static(container, out, header, max_n_seq: int = 0, status=None, stream=None) -> None:
    """aceapex_decode_all_static: the whole decode enqueued by one call that allocates nothing (the kernels' scratch
    is a static device array of the library; at most STATIC_MAX_BLOCKS blocks; calls that overlap on the GPU race).
    `container` / `out` / `status` (32 bytes, optional) are CUDA uint8 tensors, `header` the container's first 64
    bytes on the host (bytes or a numpy array)."""
    import torch
    hdr = np.ascontiguousarray(np.frombuffer(bytes(header[:64]), dtype=np.uint8))
    if hdr.size != 64:
        raise ValueError("header: the container's first 64 bytes")
    with torch.cuda.device(container.device):
        _check(lib().aceapex_decode_all_static(container.data_ptr(), container.numel(), hdr.ctypes.data, int(max_n_seq),
                                               out.data_ptr(), out.numel(), status.data_ptr() if status is not None else None,
                                               _stream_ptr(stream)), "aceapex_decode_all_static")
