"""Seeded synthetic workloads (BASELINE.json ``configs[0..4]``).

The paper measures on real FASTQ NA12878, a repetitive genome, enwik9 and silesia
(PAPER.md:65-68); none is available, so these generators take their *shapes* and stand in for
them (recipe in DESIGN.md). This module holds no codec arithmetic and is the only code that the
oracle side (tests, bench input preparation) and the CUDA side both consume.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
import threading
from dataclasses import dataclass

import numpy as np

_DIR = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_DIR, "libaceapex_workloads.so")
_SRC = os.path.join(_DIR, "gen.c")
_lock = threading.Lock()
_lib = None

KINDS = {"markov": 0, "fastq": 1, "genome": 2, "text": 3, "random": 4, "mixed": 5}
SEED_BASE = 0xACEA9E00
MIB = 1 << 20


def build(force: bool = False) -> str:
    if not force and os.path.exists(_SO) and os.path.getmtime(_SO) >= os.path.getmtime(_SRC):
        return _SO
    tmp = _SO + f".tmp{os.getpid()}"
    subprocess.run(["gcc", "-std=c11", "-O2", "-fPIC", "-shared", "-Wall", "-Wextra", "-o", tmp, _SRC, "-lm"],
                   check=True, cwd=_DIR)
    os.replace(tmp, _SO)
    return _SO


def _get():
    global _lib
    with _lock:
        if _lib is None:
            L = C.CDLL(build())
            L.aceapex_workload_generate.argtypes = [C.c_int, C.c_uint64, C.c_void_p, C.c_size_t]
            L.aceapex_workload_generate.restype = C.c_int
            _lib = L
    return _lib


def generate(kind: str, nbytes: int, seed: int) -> np.ndarray:
    """``nbytes`` of profile ``kind`` ('markov', 'fastq', 'genome', 'text', 'random', 'mixed')."""
    out = np.empty(max(1, nbytes), dtype=np.uint8)
    rc = _get().aceapex_workload_generate(KINDS[kind], seed & 0xFFFFFFFFFFFFFFFF, out.ctypes.data_as(C.c_void_p), nbytes)
    if rc != 0:
        raise ValueError(f"workload generator failed for kind={kind}")
    return out[:nbytes]


@dataclass(frozen=True)
class Config:
    """One BASELINE.json config: the data recipe plus the encoder policy it is run with."""
    name: str
    kind: str
    nbytes: int
    seed: int
    offset_width: int
    encoder: dict          # oracle encoder parameters (policy; readings A12, A15)
    stands_in_for: str

    def data(self, nbytes: int | None = None) -> np.ndarray:
        return generate(self.kind, self.nbytes if nbytes is None else nbytes, self.seed)


# Encoder policies. `literal` is the north_star wording taken literally (accept every match of
# >= 4 bytes, no scheduling promises); `scheduled` is the policy the large configs run with
# (reading A15): threshold 8, copy depth <= 8, window of 1024 blocks, in-block copy level 1,
# and a stream is stored RAW when rANS would save less than 5 % of it (selective entropy).
# `seek_aware` (a seek needs the blocks a block copies from) bounds what one
# isolated block costs: copy depth <= 3 hops and at most 128 distinct source blocks per block, both header promises
# the validator checks (a single seek's latency follows the hops; the fan-out bound mostly helps batches, and 32
# instead of 128 would cost the genome profile half its ratio: BASELINE.md). `long` adds the 12-byte long hash of SURVEY.md reading A14 (genome: the "match-dominated"
# config; 3x the encode time, so the other configs keep the short hash).
POLICY_LITERAL = dict(min_match=4, chain_depth=32, max_depth=0, window=0)
# `max_seq`: at most that many sequences per block (the rest of a dense block stays literal). The match kernel sizes
# every CTA's tables for the densest block of a container; 1536 (4-byte offsets) resp. 1344 (8-byte) keeps four CTAs
# resident per SM, and touches about one block in a hundred.
POLICY_SCHEDULED = dict(min_match=8, chain_depth=32, max_depth=8, window=1024, batch=64, max_level=1, raw_slack_pct=5,
                        max_seq=1536)
POLICY_SCHEDULED_LONG = dict(POLICY_SCHEDULED, long_hash=12, long_chain=16, max_seq=1344)
POLICY_SEEK_AWARE = dict(POLICY_SCHEDULED, max_depth=3, max_fanout=128)
POLICIES = {"literal": POLICY_LITERAL, "scheduled": POLICY_SCHEDULED, "seek_aware": POLICY_SEEK_AWARE}

CONFIGS = {
    "markov_1m": Config("markov_1m", "markov", 1 * MIB, SEED_BASE + 1, 4, POLICY_LITERAL,
                        "smoke config (BASELINE.json configs[0])"),
    "fastq_64m": Config("fastq_64m", "fastq", 64 * MIB, SEED_BASE + 2, 4, POLICY_SCHEDULED,
                        "clean (real FASTQ NA12878), PAPER.md:65"),
    "genome_256m": Config("genome_256m", "genome", 256 * MIB, SEED_BASE + 3, 8, POLICY_SCHEDULED_LONG,
                          "repeat (repetitive genome), PAPER.md:66"),
    "text_256m": Config("text_256m", "text", 256 * MIB, SEED_BASE + 4, 4, POLICY_SCHEDULED,
                        "enwik9 (English text), PAPER.md:67"),
    "mixed_1g": Config("mixed_1g", "mixed", 1024 * MIB, SEED_BASE + 5, 4, POLICY_SCHEDULED,
                       "silesia (mixed), PAPER.md:68"),
}
CONFIG_ORDER = ["markov_1m", "fastq_64m", "genome_256m", "text_256m", "mixed_1g"]


def seek_ids(n_blocks: int, count: int, seed: int) -> np.ndarray:
    """``count`` uniformly random block ids (duplicates allowed), seeded (splitmix64)."""
    ids = np.empty(count, dtype=np.uint64)
    s = np.uint64(seed & 0xFFFFFFFFFFFFFFFF)
    with np.errstate(over="ignore"):
        idx = np.arange(1, count + 1, dtype=np.uint64)
        z = s + idx * np.uint64(0x9E3779B97F4A7C15)
        z = (z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)
        z = (z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)
        z = z ^ (z >> np.uint64(31))
    ids[:] = z % np.uint64(max(1, n_blocks))
    return ids
