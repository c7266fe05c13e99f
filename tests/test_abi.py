"""CPU-side checks of the boundary (-m "not gpu"): the C-ABI library builds for sm_100a, loads, and
exports every symbol include/aceapex.h declares; argument errors are reported without a device;
the product path has no CPU fallback and never touches oracle/."""
import ctypes as C
import os
import re
import subprocess

import pytest

from conftest import ROOT

from paper_2606_24531_b200 import binding, build


def header_symbols():
    text = open(os.path.join(ROOT, "include", "aceapex.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(aceapex_[a-z_]+)\s*\(", text)))


def test_library_builds_and_exports_every_declared_symbol():
    so = build.build()
    assert os.path.exists(so)
    declared = header_symbols()
    assert declared == sorted(binding.SYMBOLS)
    nm = subprocess.run(["nm", "-D", "--defined-only", so], capture_output=True, text=True, check=True).stdout
    exported = set(re.findall(r"\bT (aceapex_[a-z_]+)\b", nm))
    assert set(declared) <= exported, sorted(set(declared) - exported)
    L = binding.lib()
    for name in declared:
        assert hasattr(L, name)


def test_library_is_sm100a_with_lineinfo_flags():
    assert "arch=compute_100a,code=sm_100a" in build.NVCC_FLAGS and "-lineinfo" in build.NVCC_FLAGS
    out = subprocess.run(["cuobjdump", "-lelf", build.build()], capture_output=True, text=True).stdout
    assert "sm_100a" in out


def test_calls_that_need_no_device():
    L = binding.lib()
    assert L.aceapex_version() >= 100
    assert L.aceapex_strerror(0) == b"ok"
    assert b"corrupt" in L.aceapex_strerror(binding.E_CORRUPT)
    ctx = C.c_void_p()
    assert L.aceapex_open(None, 100, None, C.byref(ctx)) == binding.E_ARG
    assert L.aceapex_open(16, 100, None, None) == binding.E_ARG
    assert L.aceapex_open(24, 4096, None, C.byref(ctx)) == binding.E_ARG       # misaligned device pointer
    assert L.aceapex_decode_all(None, None, 0, None) == binding.E_ARG
    assert L.aceapex_decode_range(None, 0, 1, None, 0, None) == binding.E_ARG
    assert L.aceapex_decode_blocks(None, None, 0, None, 0, 0, None) == binding.E_ARG
    assert L.aceapex_seek(None, 0, None, 0, None, None, None) == binding.E_ARG
    assert L.aceapex_scratch_bytes(None, 1, 1) == 0
    assert L.aceapex_launch_count(None) == 0
    L.aceapex_close(None)


def test_no_cpu_fallback_and_no_oracle_in_the_product():
    import torch
    if not torch.cuda.is_available():
        with pytest.raises(RuntimeError):
            binding.Decoder(b"\0" * 64)
    pkg = os.path.join(ROOT, "paper_2606_24531_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".c", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle\b", src, flags=re.M), f
                assert "aceapex_oracle" not in src and '#include "../../oracle' not in src, f
