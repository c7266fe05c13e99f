"""aceapex_decode_all_static (-m gpu): the allocation-free entry point against the existing path.

Collected last on purpose (the suite runs with pytest -x). Bar: bit-exact with Decoder.decode_all - which the other
GPU tests hold to the oracle - on calls in a row that share the library's static scratch array: a second call on
another container (stale control words, done flags and slots of the first must not leak), then the first again;
also several sub-batches, the format-maximum max_n_seq, the status words, and rejection beyond the stated maximum."""
import struct

import numpy as np
import pytest

import oracle
from paper_2606_24531_b200 import workloads as W

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu
B = 16384


@pytest.fixture(scope="module")
def binding():
    if not torch.cuda.is_available():
        pytest.fail("-m gpu tests need a CUDA device; the product has no CPU fallback")
    from paper_2606_24531_b200 import binding as b
    return b


def encode(name, nbytes, **over):
    cfg = W.CONFIGS[name]
    data = cfg.data(nbytes)
    p = dict(cfg.encoder)
    if p.get("window"):
        p.update(window=8, batch=4)
    p.update(over)
    return data, oracle.encode(data, offset_width=cfg.offset_width, threads=8, **p)


def existing_path(binding, c, n):
    with binding.Decoder(c, n_targets=1) as dec:
        out = torch.full((n,), 0xA5, dtype=torch.uint8, device="cuda")
        dec.decode_all(out)
        dec.check()
        return out, int(dec.info.max_n_seq)


def static_path(binding, c, n, max_n_seq, fill=0x5A):
    d_c = torch.from_numpy(c).cuda()
    out = torch.full((n + 64,), fill, dtype=torch.uint8, device="cuda")
    status = torch.full((32,), 0x77, dtype=torch.uint8, device="cuda")
    binding.decode_all_static(d_c, out[:n], c[:64], max_n_seq=max_n_seq, status=status)
    torch.cuda.synchronize()
    first_bad, complete, _, st, _ = struct.unpack("<QQQII", status.cpu().numpy().tobytes())
    assert torch.all(out[n:] == fill)                            # nothing beyond total_len
    return out[:n], (first_bad, complete, st)


def test_static_entry_matches_existing_path_on_calls_in_a_row(binding):
    cases = [encode("fastq_64m", 70 * B + 333), encode("text_256m", 400 * B + 5),   # 400 blocks: several sub-batches
             encode("markov_1m", 20 * B + 1)]                                       # literal policy: serial chain, deep tags
    want = []
    for data, c in cases:
        out, ms = existing_path(binding, c, data.size)
        assert np.array_equal(out.cpu().numpy(), data)
        want.append((out, ms))
    order = [0, 1, 0, 2, 1, 2, 2]                                # every call reuses the array the previous one left behind
    for i in order:
        data, c = cases[i]
        out, ms = want[i]
        nb = (data.size + B - 1) // B
        got, (first_bad, complete, st) = static_path(binding, c, data.size, ms)
        assert torch.equal(got, out), f"case {i}"
        assert (first_bad, complete, st) == (2 ** 64 - 1, nb, 0)
    # the format maximum as the bound (max_n_seq = 0): slower, same bytes
    got, (_, _, st) = static_path(binding, cases[0][1], cases[0][0].size, 0)
    assert st == 0 and torch.equal(got, want[0][0])


def test_static_entry_reports_and_rejects(binding):
    data, c = encode("fastq_64m", 8 * B)
    out, ms = existing_path(binding, c, data.size)
    # a bound below the real densest block: those blocks are left unwritten and reported, nothing else is touched
    got, (first_bad, _, st) = static_path(binding, c, data.size, 16)
    assert st != 0 and first_bad < 8
    # ... and the next call is clean again
    got, (first_bad, complete, st) = static_path(binding, c, data.size, ms)
    assert st == 0 and complete == 8 and torch.equal(got, out)
    d_c = torch.from_numpy(c).cuda()
    o = torch.empty(data.size, dtype=torch.uint8, device="cuda")
    with pytest.raises(binding.AceapexError) as e:               # output too small
        binding.decode_all_static(d_c, o[:-1], c[:64], max_n_seq=ms)
    assert e.value.code == binding.E_CAPACITY
    bad = c[:64].copy(); bad[0] = ord("X")
    with pytest.raises(binding.AceapexError) as e:
        binding.decode_all_static(d_c, o, bad, max_n_seq=ms)
    assert e.value.code == binding.E_FORMAT
    # beyond the stated maximum of 4,096 blocks: a clear error, nothing enqueued
    big = W.generate("random", (binding.STATIC_MAX_BLOCKS + 1) * B, 3)
    cb = oracle.encode(big, min_match=B, threads=8)              # literals only: quick to encode
    d_cb = torch.from_numpy(cb).cuda()
    ob = torch.full((big.size,), 0xA5, dtype=torch.uint8, device="cuda")
    with pytest.raises(binding.AceapexError) as e:
        binding.decode_all_static(d_cb, ob, cb[:64], max_n_seq=16)
    assert e.value.code == binding.E_CAPACITY
    torch.cuda.synchronize()
    assert torch.all(ob == 0xA5)
    # exactly the maximum is accepted (random bytes: every block a straight literal copy)
    okd = big[: binding.STATIC_MAX_BLOCKS * B]
    co = oracle.encode(okd, min_match=B, threads=8)
    got, (_, complete, st) = static_path(binding, co, okd.size, 16)
    assert st == 0 and complete == binding.STATIC_MAX_BLOCKS and np.array_equal(got.cpu().numpy(), okd)
