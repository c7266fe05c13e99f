"""Run by tests/test_gpu_blocksize.py in its own interpreter with ACEAPEX_BLOCK_LOG2 and ACEAPEX_LIB set: the CUDA
library variant of that block size against the oracle variant of the same size, bit for bit (decode_all vs decoder #1,
isolated blocks vs decoder #2, a range, the hand-made container of the independent writer)."""
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
sys.path.insert(0, os.path.join(ROOT, "tests"))

import numpy as np
import torch

import oracle
from paper_2606_24531_b200 import binding, workloads as W
from handmade import B, container_from_tokens, expand
from test_oracle_codec import handmade_case

assert oracle.B == binding.B == B == 1 << int(os.environ["ACEAPEX_BLOCK_LOG2"])
BL = oracle.BLOG


def check(c, want, n_targets=8):
    n = want.size
    with binding.Decoder(c, n_targets=n_targets) as dec, oracle.Isolated(c) as iso:
        assert dec.info.block_size == B and dec.info.total_len == n
        out = torch.full((n + 64,), 0xA5, dtype=torch.uint8, device="cuda")
        dec.decode_all(out); dec.check()
        got = out.cpu().numpy()
        assert np.array_equal(got[:n], want) and np.all(got[n:] == 0xA5)
        nb = int(dec.info.n_blocks)
        rng = np.random.default_rng(5)
        ids = sorted(set([0, nb // 2, nb - 1] + [int(x) for x in rng.integers(0, nb, 12)]))
        got = dec.decode_blocks(np.array(ids, np.uint64), torch.full((len(ids) * B,), 0xA5, dtype=torch.uint8, device="cuda")).cpu().numpy()
        dec.check()
        for i, b in enumerate(ids):
            blk = iso.decode(b)
            assert np.array_equal(got[i * B:i * B + blk.size], blk), b
            assert np.all(got[i * B + blk.size:(i + 1) * B] == 0xA5)
        blk, start, blen = dec.seek((nb - 1) * B + 1)
        assert start == (nb - 1) * B and np.array_equal(blk.cpu().numpy()[:blen], iso.decode(nb - 1))
        if nb >= 6:
            first, cnt = nb // 3, nb // 3
            r = torch.full((cnt * B,), 0xA5, dtype=torch.uint8, device="cuda")
            dec.decode_range(first, cnt, r); dec.check()
            assert np.array_equal(r.cpu().numpy(), want[first * B:(first + cnt) * B])


total, blocks = handmade_case()
check(container_from_tokens(total, blocks), np.frombuffer(expand(total, blocks), np.uint8), n_targets=3)
for name, pol in (("text_256m", "scheduled"), ("fastq_64m", "scheduled"), ("markov_1m", "literal"), ("mixed_1g", "scheduled")):
    cfg = W.CONFIGS[name]
    data = cfg.data(40 * B + 777)
    p = dict(W.POLICIES[pol])
    if p.get("window"):
        p.update(window=6, batch=4)
    if p.get("max_seq"):
        p["max_seq"] = max(16, (p["max_seq"] << BL) >> 14)
    c = oracle.encode(data, offset_width=cfg.offset_width, threads=4, **p)
    want = oracle.decode_all(c)
    assert np.array_equal(want, data)
    check(c, want)
print("blocksize check ok", B)
