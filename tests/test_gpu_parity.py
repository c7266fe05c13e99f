"""Parity of the CUDA path against the CPU oracle (-m gpu), through the C-ABI.

Bar: bit-exact. Every byte of decode_all against oracle decoder #1; every isolated block against
oracle decoder #2; the entropy layer on its own against the oracle's per-stream decode
(PAPER.md:41 checks the ANS round trip separately); the paper's three-phase isolation check
 with the untouched check extended to the whole buffer and a non-zero fill
("empty-buffer trap"). Inputs are seeded and synthetic (DESIGN.md recipe).
"""
import ctypes as C

import numpy as np
import pytest

import oracle
from paper_2606_24531_b200 import workloads as W

from handmade import B, build_container, build_record, container_from_tokens, expand
from test_oracle_codec import ADVERSARIAL, handmade_case

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def binding():
    if not torch.cuda.is_available():
        pytest.fail("-m gpu tests need a CUDA device; the product has no CPU fallback")
    from paper_2606_24531_b200 import binding as b
    return b


def dev_out(n, fill=0xA5):
    return torch.full((max(1, n),), fill, dtype=torch.uint8, device="cuda")


def full_check(binding, c, want, n_slots=None, n_targets=16, seek_blocks=None, fills=(0xA5,)):
    """decode_all == want; listed (default: all) blocks decode in isolation to want's ranges."""
    want = np.frombuffer(want, np.uint8) if isinstance(want, (bytes, bytearray)) else want
    n = want.size
    with binding.Decoder(c, n_slots=n_slots, n_targets=n_targets) as dec:
        assert dec.info.total_len == n
        for fill in fills:
            out = dev_out(n + 64, fill)
            dec.decode_all(out)
            dec.check()
            got = out.cpu().numpy()
            assert np.array_equal(got[:n], want)
            assert np.all(got[n:] == fill)                       # nothing beyond total_len
        nb = int(dec.info.n_blocks)
        ids = list(range(nb)) if seek_blocks is None else list(seek_blocks)
        if ids:
            got = dec.decode_blocks(np.array(ids, np.uint64), dev_out(len(ids) * B)).cpu().numpy()
            dec.check()
            for i, b in enumerate(ids):
                blen = min(B, n - b * B)
                assert np.array_equal(got[i * B:i * B + blen], want[b * B:b * B + blen]), b
                assert np.all(got[i * B + blen:(i + 1) * B] == 0xA5)
        return dec.launch_count


# ------------------------------------------------------------------ configs (BASELINE.json configs[0..4])

def test_config0_markov_1m_decode_all_and_seek_every_block(binding):
    cfg = W.CONFIGS["markov_1m"]
    data = cfg.data()
    c = oracle.encode(data, offset_width=cfg.offset_width, threads=4, **cfg.encoder)
    want = oracle.decode_all(c)
    assert np.array_equal(want, data)
    assert oracle.info(c).max_depth == 0                         # literal policy: no depth promise -> read-back hop loop
    full_check(binding, c, want, fills=(0x00, 0xA5))
    # every block through aceapex_seek, compared with oracle decoder #2
    with binding.Decoder(c, n_targets=1) as dec, oracle.Isolated(c) as iso:
        for b in range(int(dec.info.n_blocks)):
            blk, start, blen = dec.seek(b * B + (b * 37) % B)
            assert (start, blen) == (b * B, B)
            assert np.array_equal(blk.cpu().numpy()[:blen], iso.decode(b)), b
        dec.check()


SAMPLES = [("fastq_64m", 6 << 20), ("genome_256m", 6 << 20), ("text_256m", 6 << 20), ("mixed_1g", 6 << 20)]


@pytest.mark.parametrize("name,nbytes", SAMPLES)
@pytest.mark.parametrize("policy", ["scheduled", "literal", "seek_aware"])
def test_profile_samples_bit_exact(binding, name, nbytes, policy):
    """Several hundred blocks of each profile, ragged tail, under the three encoder policies (seek_aware: the
    config's own policy with the copy-depth and fan-out bounds of SURVEY.md section 8f rank 4 and a low max_seq)."""
    cfg = W.CONFIGS[name]
    nbytes += 12345                                              # ragged last block
    data = cfg.data(nbytes)
    params = dict(cfg.encoder) if policy != "literal" else dict(W.POLICY_LITERAL)
    if policy == "seek_aware":
        params.update(max_depth=W.POLICY_SEEK_AWARE["max_depth"], max_fanout=6, max_seq=700)
    if params.get("window"):
        params.update(window=24, batch=8)                        # scaled so that cross-block matches exist
    c = oracle.encode(data, offset_width=cfg.offset_width, threads=8, **params)
    want = oracle.decode_all(c)
    nb = oracle.info(c).n_blocks
    rng = np.random.default_rng(7)
    ids = sorted(set([0, 1, nb // 2, nb - 2, nb - 1] + [int(x) for x in rng.integers(0, nb, 24)]))
    full_check(binding, c, want, seek_blocks=ids, n_targets=8)
    with binding.Decoder(c, n_targets=4) as dec, oracle.Isolated(c) as iso:
        for b in ids[:6] + ids[-2:]:
            blk, start, blen = dec.seek(b * B + 1)
            assert np.array_equal(blk.cpu().numpy()[:blen], iso.decode(b)), b
        dec.check()


def test_bench_config_fastq_64m_full_size(binding):
    """BASELINE.json configs[1] at full size in the launch configuration bench.py times."""
    cfg = W.CONFIGS["fastq_64m"]
    data = cfg.data()
    c = oracle.encode(data, offset_width=cfg.offset_width, threads=8, **cfg.encoder)
    want = oracle.decode_all(c)
    assert oracle.fnv1a64(want) == oracle.fnv1a64(data)
    nb = oracle.info(c).n_blocks
    ids = [int(x) for x in W.seek_ids(nb, 48, W.SEED_BASE + 0x72)] + [0, nb - 1]
    full_check(binding, c, want, seek_blocks=ids, n_targets=64)


@pytest.mark.parametrize("name", ["genome_256m", "text_256m"])
def test_configs_2_3_full_size(binding, name):
    """BASELINE.json configs[2] (8-byte offsets) and configs[3] at full size (16,384 blocks): decode_all against
    the original bytes (round-trip identity pins the oracle), sampled isolated blocks against oracle decoder #2."""
    cfg = W.CONFIGS[name]
    data = cfg.data()
    c = oracle.encode(data, offset_width=cfg.offset_width, threads=8, **cfg.encoder)
    assert oracle.info(c).offset_width == cfg.offset_width
    nb = int(oracle.info(c).n_blocks)
    ids = [int(x) for x in W.seek_ids(nb, 24, W.SEED_BASE + 0x73)] + [0, nb - 1]
    with binding.Decoder(c, n_targets=32) as dec, oracle.Isolated(c) as iso:
        out = dev_out(data.size)
        dec.decode_all(out)
        dec.check()
        assert torch.equal(out.cpu(), torch.from_numpy(data))
        got = dec.decode_blocks(np.array(ids, np.uint64), dev_out(len(ids) * B)).cpu().numpy()
        dec.check()
        for i, b in enumerate(ids):
            blk = iso.decode(b)
            assert np.array_equal(got[i * B:i * B + blk.size], blk), b


def test_config4_mixed_1g_full_size(binding):
    """BASELINE.json configs[4] at full size with the binding's defaults (one batch of 65,536 slots): decode_all
    against the original bytes (round-trip identity pins decoder #1); the seeded 100,000 block ids as ONE
    decode_blocks(PACKED) at n_targets=1024 (the group size bench.py times), every block compared with the original
    (decoder #2 == decoder #1 == original is pinned on the CPU side); 2,048 individual aceapex_seek calls compared the
    same way and 48 of them against oracle decoder #2 itself."""
    cfg = W.CONFIGS["mixed_1g"]
    data = cfg.data()
    c = oracle.encode(data, offset_width=cfg.offset_width, threads=32, **cfg.encoder)
    nb = int(oracle.info(c).n_blocks)
    assert nb == 65536
    d_data = torch.from_numpy(data).cuda()
    with binding.Decoder(c, n_targets=1024) as dec:
        assert dec.n_slots == 65536
        out = dev_out(data.size)
        dec.decode_all(out)
        dec.check()
        assert torch.equal(out, d_data)
        del out
        ids = W.seek_ids(nb, 100_000, W.SEED_BASE + 0x70 + 4)
        bout = dev_out(len(ids) * B)
        dec.decode_blocks(ids, bout)
        dec.check()
        idx = torch.from_numpy(ids.astype(np.int64)).cuda()
        step = 10_000                                               # compare in slices: keeps the gather small
        for i in range(0, len(ids), step):
            want = d_data.view(nb, B)[idx[i:i + step]]
            assert torch.equal(bout.view(-1, B)[i:i + step], want), i
        del bout
        dst = dev_out(B)
        with oracle.Isolated(c) as iso:
            for j, b in enumerate(ids[:2048]):
                b = int(b)
                _, start, blen = dec.seek(b * B + (j * 131) % B, dst)
                assert (start, blen) == (b * B, B)
                assert torch.equal(dst, d_data[b * B:(b + 1) * B]), b
                if j < 48:
                    assert np.array_equal(dst.cpu().numpy(), iso.decode(b)), b
        dec.check()


# ------------------------------------------------------------------ entropy layer alone

@pytest.mark.parametrize("name", ["markov_1m", "genome_256m"])
def test_entropy_layer_streams_match_oracle(binding, name):
    cfg = W.CONFIGS[name]
    data = cfg.data(40 * B + 999)
    params = dict(cfg.encoder)
    if params.get("window"):
        params.update(window=4, batch=4)
    c = oracle.encode(data, offset_width=cfg.offset_width, **params)
    nb = oracle.info(c).n_blocks
    with binding.Decoder(c) as dec:
        lit, ln, off = (t.cpu().numpy() for t in dec.decode_streams(0, nb))
        dec.check()
    for b in range(nb):
        h, olit, olen, ooff, _, _ = oracle.decode_streams(c, b)
        assert np.array_equal(lit[b * B:b * B + olit.size], olit), b
        assert np.array_equal(ln[b * 8192:b * 8192 + olen.size], olen), b
        assert np.array_equal(off[b * 32768:b * 32768 + ooff.size], ooff), b


# ------------------------------------------------------------------ handmade and adversarial inputs

def test_handmade_tokens_spanning_source_escapes_deep_tags(binding):
    total, blocks = handmade_case()
    c = container_from_tokens(total, blocks)
    want = oracle.decode_all(c)
    full_check(binding, c, want, fills=(0x00, 0xA5))
    c8 = container_from_tokens(total, blocks, off_width=8)
    full_check(binding, c8, want)


@pytest.mark.parametrize("name", sorted(ADVERSARIAL))
def test_adversarial_sizes(binding, name):
    data = ADVERSARIAL[name]
    for params in (dict(min_match=4), dict(min_match=8, max_depth=3, window=2, batch=2)):
        c = oracle.encode(data, **params)
        want = oracle.decode_all(c)
        assert want.tobytes() == data
        full_check(binding, c, want)


def test_max_sequences_per_block(binding):
    """4095 sequences in one block (the most a 16 KiB block can hold: 4 literals, then 4-byte matches)."""
    lits = b"wxyz"
    seqs = [(4, 4, 0)] + [(0, 4, 0) for k in range(1, 4095)]
    blocks = [(seqs, lits)]
    c = container_from_tokens(B, blocks)
    want = oracle.decode_all(c)
    assert want.tobytes() == b"wxyz" * 4096
    full_check(binding, c, want)
    # and 4096 single-literal sequences with 255+ escapes in a second block reading the first
    seqs2 = [(1, 4, 8 * k) for k in range(2048)] + [(300, 5000, 0)]
    lits2 = bytes((k * 11) & 0xFF for k in range(2048 + 300)) + b"!" * (B - (2048 * 5 + 300 + 5000))
    c2 = container_from_tokens(2 * B, [(seqs, lits), (seqs2, lits2)])
    full_check(binding, c2, oracle.decode_all(c2))


def test_small_scratch_batches_and_slot_overflow(binding):
    """decode_all in batches of 5 slots; isolated decode with 3 slots (several passes per hop)."""
    data = W.generate("text", 40 * B + 17, 77)
    for params in (dict(min_match=4), dict(min_match=8, max_depth=4, window=3, batch=3)):
        c = oracle.encode(data, **params)
        want = oracle.decode_all(c)
        full_check(binding, c, want, n_slots=5, n_targets=2, seek_blocks=[40, 39, 17, 17, 3, 0])
        full_check(binding, c, want, n_slots=3, n_targets=1, seek_blocks=[33, 40])


def test_multi_boundary_group_with_source_at_position_zero(binding):
    """A 4-byte output group with two run boundaries whose last run is a match from absolute position 0: the
    word-granular gather must not touch the bytes in front of the output buffer (the buffer is a fresh allocation)."""
    lits0 = bytes((i * 13 + 1) & 0xFF for i in range(B))
    # block 1: match(4) from 100 | 1 literal | match(4) from 0 | 2 literals | match(5) from 1 | rest literals
    seqs1 = [(0, 4, 100), (1, 4, 0), (2, 5, 1), (1, 4, 0), (1, 4, 1)]
    nlit1 = B - sum(ml for _, ml, _ in seqs1)
    lits1 = bytes((i * 7 + 5) & 0xFF for i in range(nlit1))
    blocks = [([], lits0), (seqs1, lits1)]
    want = np.frombuffer(expand(2 * B, blocks), np.uint8)
    c = container_from_tokens(2 * B, blocks)
    assert np.array_equal(oracle.decode_all(c), want)
    torch.cuda.empty_cache()
    with binding.Decoder(c, n_targets=2) as dec:
        out = torch.full((64 << 20,), 0xA5, dtype=torch.uint8, device="cuda")   # its own segment: nothing mapped in front is ours
        dec.decode_all(out)
        dec.check()
        assert np.array_equal(out[:2 * B].cpu().numpy(), want)
        assert bool((out[2 * B:] == 0xA5).all())
        got = dec.decode_blocks(np.array([1, 0], np.uint64), dev_out(2 * B)).cpu().numpy()
        dec.check()
        assert np.array_equal(got[:B], want[B:]) and np.array_equal(got[B:], want[:B])


def test_two_open_decoders_of_different_containers(binding):
    """Two live contexts whose containers need different amounts of match-kernel shared memory (config 0 under the
    literal policy has thousands of sequences per block, FASTQ a few hundred) must not disturb each other."""
    big = W.CONFIGS["markov_1m"].data(8 * B)
    c_big = oracle.encode(big, **W.POLICY_LITERAL)
    small = W.generate("fastq", 8 * B + 5, 3)
    c_small = oracle.encode(small, min_match=8, max_depth=8, window=2, batch=2)
    with binding.Decoder(c_big, n_targets=2) as d_big:
        o1 = dev_out(big.size)
        d_big.decode_all(o1); d_big.check()
        with binding.Decoder(c_small, n_targets=2) as d_small:
            assert d_small.info.max_n_seq < d_big.info.max_n_seq
            o2 = dev_out(small.size)
            d_small.decode_all(o2); d_small.check()
            o1.fill_(0xA5)
            d_big.decode_all(o1); d_big.check()                  # after the smaller container was opened
            o2.fill_(0xA5)
            d_small.decode_all(o2); d_small.check()
            assert np.array_equal(o2.cpu().numpy(), small)
        assert np.array_equal(o1.cpu().numpy(), big)


def test_rejects_inconsistent_tag(binding):
    """FORMAT.md section 4: tag 0 iff the source range lies entirely below the block. A match tagged 0 whose source
    reaches into its own block (it would read bytes that pass 0 has not produced yet) is reported, not decoded."""
    lits = b"abcdefgh" + b"z" * (B - 16)
    rec = build_record(0, [(8, 8, 0)], lits, tags=[0])              # in-block source, tag says cross-block
    with binding.Decoder(build_container(B, [rec]), n_targets=1) as dec:
        out = dev_out(B + 64)
        dec.decode_all(out)
        rc, first = dec.device_status(clear=True)
        assert rc == binding.E_CORRUPT and first == 0
        assert bool((out == 0xA5).all())                             # the bad block is left unwritten
        # the isolated path never uses tags (scheduling metadata): it returns the right bytes
        got = dec.decode_blocks(np.array([0], np.uint64), dev_out(B)).cpu().numpy()
        assert dec.device_status()[0] == 0 and got[:16].tobytes() == b"abcdefghabcdefgh"
    lits0 = bytes(range(256)) * (B // 256)
    rec0 = build_record(0, [], lits0)
    rec1 = build_record(B, [(8, 8, 16)], lits, tags=[1])            # source entirely below the block, tag says in-block
    with binding.Decoder(build_container(2 * B, [rec0, rec1]), n_targets=1) as dec:
        dec.decode_all(dev_out(2 * B))
        rc, first = dec.device_status(clear=True)
        assert rc == binding.E_CORRUPT and first == 1


# ------------------------------------------------------------------ range decode

def check_range(binding, dec, want, first, count, fill=0xA5):
    """decode_range(first, count) into a guarded range-sized buffer == want's bytes; nothing outside is written."""
    n = want.size
    lo, hi = first * B, min(n, (first + count) * B)
    guard = 4096
    buf = dev_out(guard + count * B + guard, fill)
    dec.decode_range(first, count, buf[guard:])
    dec.check()
    got = buf.cpu().numpy()
    assert np.array_equal(got[guard:guard + hi - lo], want[lo:hi]), (first, count)
    assert np.all(got[:guard] == fill) and np.all(got[guard + hi - lo:] == fill), (first, count)


@pytest.mark.parametrize("policy", ["scheduled", "literal", "small_window"])
def test_range_decode_samples(binding, policy):
    """Ranges at the start, in the middle and at the ragged end of a text sample under three encoder policies: with
    the literal policy and the small window most cross-block sources of a mid-file range lie INSIDE the range (match
    kernel), with the scheduled window all of them lie below it (isolated chase); sub-batches smaller than the range."""
    data = W.generate("text", 150 * B + 4321, 91)
    params = {"scheduled": dict(min_match=8, max_depth=8, window=64, batch=8, max_level=1, raw_slack_pct=5),
              "literal": dict(W.POLICY_LITERAL), "small_window": dict(min_match=6, max_depth=6, window=3, batch=3)}[policy]
    c = oracle.encode(data, threads=8, **params)
    want = oracle.decode_all(c)
    assert np.array_equal(want, data)
    nb = int(oracle.info(c).n_blocks)
    with binding.Decoder(c, n_targets=64) as dec:
        for first, count in ((0, 40), (0, nb), (1, 1), (37, 50), (100, nb - 100), (nb - 1, 1), (70, 3)):
            check_range(binding, dec, want, first, count)
        L = binding.lib()
        buf = dev_out(4 * B)
        assert L.aceapex_decode_range(dec._ctx, nb - 1, 2, buf.data_ptr(), buf.numel(), None) == binding.E_RANGE
        assert L.aceapex_decode_range(dec._ctx, 5, 4, buf.data_ptr(), 4 * B - 1, None) == binding.E_CAPACITY
        assert L.aceapex_decode_range(dec._ctx, 5, 0, None, 0, None) == 0
    with binding.Decoder(c, n_slots=7, n_targets=5) as dec:          # sub-batches of 5 blocks
        check_range(binding, dec, want, 60, 23)
        check_range(binding, dec, want, 0, 23)
    with binding.Decoder(c, n_targets=0) as dec:                     # no isolated scratch: only ranges from block 0
        check_range(binding, dec, want, 0, 30)
        buf = dev_out(2 * B)
        assert binding.lib().aceapex_decode_range(dec._ctx, 3, 2, buf.data_ptr(), buf.numel(), None) == binding.E_STATE


def test_range_decode_handmade_spanning_and_deep(binding):
    """The handmade container (a source that spans two blocks, tags 1..11, escapes): every range of it."""
    total, blocks = handmade_case()
    c = container_from_tokens(total, blocks)
    want = np.frombuffer(expand(total, blocks), np.uint8)
    with binding.Decoder(c, n_targets=2) as dec:
        for first in range(3):
            for count in range(1, 4 - first):
                check_range(binding, dec, want, first, count, fill=0x00)
                check_range(binding, dec, want, first, count)


def test_range_decode_text_256m_blocks_0_1000_and_mid_file(binding):
    """SURVEY.md section 8(f)-2 / PAPER.md:104: blocks 0-1000 and a mid-file range of 1,001 blocks of configs[3]
    into a 1,001-block buffer, bit-exact against the original bytes (= decoder #1), nothing written outside."""
    cfg = W.CONFIGS["text_256m"]
    data = cfg.data()
    c = oracle.encode(data, offset_width=cfg.offset_width, threads=32, **cfg.encoder)
    nb = int(oracle.info(c).n_blocks)
    with binding.Decoder(c, n_targets=1024) as dec:
        check_range(binding, dec, data, 0, 1001)
        check_range(binding, dec, data, nb // 2, 1001)
        check_range(binding, dec, data, nb - 1001, 1001)
        check_range(binding, dec, data, 5000, 3000)                  # three sub-batches of 1,024 targets


# ------------------------------------------------------------------ isolation

@pytest.mark.parametrize("fill", [0x00, 0xA5])
def test_three_phase_isolation(binding, fill):
    data = W.generate("fastq", 24 * B + 100, 42)
    c = oracle.encode(data, min_match=8, max_depth=8, window=2, batch=2)
    n = data.size
    with binding.Decoder(c, n_targets=4) as dec:
        for target in (0, 7, 23, 24):
            buf = dev_out(n, fill)
            lo, hi = target * B, min(n, (target + 1) * B)
            assert oracle.fnv1a64(buf[lo:hi].cpu().numpy()) != oracle.fnv1a64(data[lo:hi])      # phase 1
            dec.decode_blocks(np.array([target], np.uint64), buf, flags=binding.ABSOLUTE)
            dec.check()
            got = buf.cpu().numpy()
            assert oracle.fnv1a64(got[lo:hi]) == oracle.fnv1a64(data[lo:hi])                     # phase 2
            assert np.array_equal(got[lo:hi], data[lo:hi])
            mask = np.ones(n, bool); mask[lo:hi] = False
            assert np.all(got[mask] == fill)                                                     # phase 3: whole buffer
        # aceapex_seek writes only block_len bytes of its destination
        dst = dev_out(B + 32, fill)
        _, start, blen = dec.seek(n - 1, dst)
        assert (start, blen) == (24 * B, 100)
        got = dst.cpu().numpy()
        assert np.array_equal(got[:100], data[24 * B:]) and np.all(got[100:] == fill)


def test_decode_blocks_absolute_duplicates_and_errors(binding):
    data = W.generate("genome", 9 * B + 5, 11)
    c = oracle.encode(data, min_match=8, max_depth=6, window=2, batch=2, offset_width=8)
    with binding.Decoder(c, n_targets=3) as dec:
        buf = dev_out(data.size)
        ids = np.array([9, 2, 2, 5, 9, 0, 2], np.uint64)
        dec.decode_blocks(ids, buf, flags=binding.ABSOLUTE)
        dec.check()
        got = buf.cpu().numpy()
        for b in range(10):
            lo, hi = b * B, min(data.size, (b + 1) * B)
            if b in (0, 2, 5, 9):
                assert np.array_equal(got[lo:hi], data[lo:hi])
            else:
                assert np.all(got[lo:hi] == 0xA5)
        L = binding.lib()
        one = np.array([10], np.uint64)
        assert L.aceapex_decode_blocks(dec._ctx, one.ctypes.data_as(C.c_void_p), 1, buf.data_ptr(), buf.numel(), 0, None) == binding.E_RANGE
        assert L.aceapex_seek(dec._ctx, data.size, buf.data_ptr(), buf.numel(), None, None, None) == binding.E_RANGE
        assert L.aceapex_seek(dec._ctx, 0, buf.data_ptr(), 100, None, None, None) == binding.E_CAPACITY
        assert L.aceapex_decode_all(dec._ctx, buf.data_ptr(), data.size - 1, None) == binding.E_CAPACITY
        two = np.array([0, 1], np.uint64)
        assert L.aceapex_decode_blocks(dec._ctx, two.ctypes.data_as(C.c_void_p), 2, buf.data_ptr(), 2 * B - 1, 0, None) == binding.E_CAPACITY
        assert L.aceapex_decode_blocks(dec._ctx, two.ctypes.data_as(C.c_void_p), 2, buf.data_ptr(), buf.numel(), 7, None) == binding.E_ARG


def test_unaligned_output_pointer(binding):
    data = W.generate("text", 5 * B + 3, 5)
    c = oracle.encode(data, min_match=4)
    with binding.Decoder(c) as dec:
        buf = dev_out(data.size + 16)
        dec.decode_all(buf[3:])
        dec.check()
        got = buf.cpu().numpy()
        assert np.all(got[:3] == 0xA5) and np.array_equal(got[3:3 + data.size], data)
        assert np.all(got[3 + data.size:] == 0xA5)


# ------------------------------------------------------------------ invalid containers

def open_rc(binding, c):
    t = torch.from_numpy(np.ascontiguousarray(c)).cuda()
    ctx = C.c_void_p()
    rc = binding.lib().aceapex_open(t.data_ptr(), t.numel(), None, C.byref(ctx))
    if rc == 0:
        binding.lib().aceapex_close(ctx)
    return rc


def test_rejects_bad_header_fields(binding):
    c = oracle.encode(b"hello hello hello hello")
    for off, val in ((0, ord("X")), (8, 2), (12, 15), (13, 5), (14, 16), (15, 11)):
        bad = c.copy(); bad[off] = val
        assert open_rc(binding, bad) == binding.E_FORMAT
    assert open_rc(binding, c[:48].copy()) == binding.E_FORMAT
    assert open_rc(binding, c[:-16].copy()) == binding.E_FORMAT
    assert open_rc(binding, c) == 0


def expect_corrupt(binding, c, n, bad_block=None):
    """The device reports CORRUPT, leaves the bad block unwritten and never writes out of bounds."""
    with binding.Decoder(c, n_targets=2) as dec:
        out = dev_out(n + 4096)
        dec.decode_all(out)
        rc, first = dec.device_status(clear=True)
        assert rc == binding.E_CORRUPT
        got = out.cpu().numpy()
        assert np.all(got[n:] == 0xA5)
        if bad_block is not None:
            assert first == bad_block
            assert np.all(got[bad_block * B:min(n, (bad_block + 1) * B)] == 0xA5)
        assert dec.device_status()[0] == 0                       # cleared
        buf = dev_out(B + 64)
        dec.decode_blocks(np.array([bad_block or 0], np.uint64), buf)
        assert dec.device_status(clear=True)[0] == binding.E_CORRUPT
        assert np.all(buf.cpu().numpy()[B:] == 0xA5)


def test_rejects_overlapping_or_forward_match(binding):
    lits = b"abcdefgh" + b"z" * (B - 16)
    for src, ml in ((4, 8), (8, 8), (1 << 20, 8)):              # overlaps dst / starts at dst / beyond
        rec = build_record(0, [(8, ml, src)], lits, tags=[1])
        expect_corrupt(binding, build_container(B, [rec]), B, 0)


def test_rejects_bad_frequency_sum_state_and_token_sums(binding):
    total, blocks = handmade_case()
    good = container_from_tokens(total, blocks)
    i = oracle.info(good)
    bad = good.copy()
    bad[i.payload_off + 32 + 32] ^= 1                            # block 0 LIT table: sum != 4096
    expect_corrupt(binding, bad, total, 0)
    bad = good.copy()
    st = 64 + (i.n_blocks + 1) * 8 + (1 * 3 + 1) * 32 * 4 + 5 * 4   # block 1, LEN stream, lane 5
    bad[st] ^= 0x40
    expect_corrupt(binding, bad, total, 1)
    rec = build_record(0, [(8, 8, 0)], b"ABCDEFGH" + b"q" * 10)  # tokens do not add up to the block length
    expect_corrupt(binding, build_container(B, [rec]), B, 0)


def test_open_rejects_corrupt_record_header(binding):
    total, blocks = handmade_case()
    good = container_from_tokens(total, blocks)
    i = oracle.info(good)
    bad = good.copy()
    bad[i.payload_off + 6] = 9                                   # off_nbytes > W
    assert open_rc(binding, bad) == binding.E_CORRUPT
    bad = good.copy()
    bad[i.payload_off + 8] ^= 0x10                               # n_words[LIT] changed: section layout no longer fits
    assert open_rc(binding, bad) == binding.E_CORRUPT


def test_broken_depth_promise_does_not_affect_isolated_decode(binding):
    """The fused isolated kernel loops on the device until no byte is pending: it never relies on the
    header's depth promise D, so a container that breaks the promise still decodes bit-exactly."""
    total, blocks = handmade_case()                              # real chase depth 11
    recs = [build_record(b * B, s, l) for b, (s, l) in enumerate(blocks)]
    c = build_container(total, recs, max_depth=3)
    want = oracle.decode_all(c)
    with binding.Decoder(c, n_targets=2) as dec, oracle.Isolated(c) as iso:
        out = dev_out(total)
        dec.decode_all(out)                                      # decode_all does not rely on the promise either
        dec.check()
        assert np.array_equal(out.cpu().numpy(), want)
        nb = (total + B - 1) // B
        for b in range(nb):
            got = dec.decode_blocks(np.array([b], np.uint64), dev_out(B)).cpu().numpy()
            dec.check()
            blk = iso.decode(b)
            assert np.array_equal(got[:blk.size], blk)


# ---- selective entropy: RAW streams (FORMAT.md section 2 modes)

def test_raw_streams_handmade_and_encoder_chosen(binding):
    total, blocks = handmade_case()
    want = np.frombuffer(expand(total, blocks), np.uint8)
    for raw in [("lit",), ("len",), ("off",), ("lit", "len", "off")]:
        recs = []
        for b, (seqs, lits) in enumerate(blocks):
            use = tuple(k for k in raw if not (k == "lit" and len(lits) == 0))
            recs.append(build_record(b * B, seqs, lits, raw=use))
        full_check(binding, build_container(total, recs), want, n_targets=2)
    # encoder-chosen: uniform random bytes (LIT raw in every block) and a high slack (everything raw)
    rnd = W.generate("random", 5 * B + 77, 11)
    c, st = oracle.encode(rnd, return_stats=True)
    assert st.n_raw[0] == 6
    full_check(binding, c, rnd, n_targets=3)
    fq = W.generate("fastq", 24 * B + 5, 12)
    c, st = oracle.encode(fq, return_stats=True, min_match=8, max_depth=8, window=4, batch=4, raw_slack_pct=1000)
    assert sum(st.n_raw) >= 2 * 25
    full_check(binding, c, fq, n_targets=5, seek_blocks=[0, 24, 7, 19, 13, 3])


def test_rejects_inconsistent_raw_streams(binding):
    total, blocks = handmade_case()
    recs = [build_record(b * B, s, l, raw=("len",)) for b, (s, l) in enumerate(blocks)]
    good = build_container(total, recs)
    i = oracle.info(good)
    bad = good.copy(); bad[i.payload_off + 7] = 0x0C                      # reserved mode 3 for LEN
    assert open_rc(binding, bad) == binding.E_CORRUPT
    bad = good.copy(); bad[i.payload_off + 7] = 0x08                      # CONST for LEN, but its n_words is not 1
    assert open_rc(binding, bad) == binding.E_CORRUPT
    bad = good.copy(); bad[i.payload_off + 8 + 4] ^= 1                    # n_words[LEN] != ceil(n_sym / 2)
    assert open_rc(binding, bad) == binding.E_CORRUPT
    bad = good.copy()
    st = 64 + (i.n_blocks + 1) * 8 + (1 * 3 + 1) * 32 * 4 + 7 * 4         # block 1, LEN stream, lane 7
    bad[st] ^= 1                                                          # an unused state that is not 2^16
    expect_corrupt(binding, bad, total, 1)
    rec, stt = build_record(0, [], b"abc", raw=("lit",))
    c = build_container(3, [(rec, stt)])
    full_check(binding, c, np.frombuffer(b"abc", np.uint8), n_targets=1)
    bad = c.copy(); bad[oracle.info(c).payload_off + 32 + 3] = 1          # pad byte of the odd raw stream
    expect_corrupt(binding, bad, 3, 0)


def test_const_streams_handmade_and_encoder_chosen(binding):
    """CONST stream mode (FORMAT.md section 2 mode 2): containers whose LIT / LEN / OFF streams are constant by
    construction (tests/test_oracle_codec.py const_case), the encoder's own choice on equal bytes, malformed records."""
    from test_oracle_codec import const_case
    total, blocks = const_case()
    want = np.frombuffer(expand(total, blocks), np.uint8)
    for const in [("lit",), ("len",), ("off",), ("lit", "len", "off")]:
        recs = []
        for b, (seqs, lits) in enumerate(blocks):
            use = tuple(k for k in const if k == "lit" or seqs)
            recs.append(build_record(b * B, seqs, lits, const=use))
        full_check(binding, build_container(total, recs), want, n_targets=2)
    data = np.frombuffer(ADVERSARIAL["all_equal"], np.uint8)
    c, st = oracle.encode(data, return_stats=True)
    assert sum(st.n_const) >= 1
    full_check(binding, c, data, n_targets=2)
    # malformed: a state that is not 2^16, a non-zero high byte of the word
    recs = [build_record(b * B, s, l, const=("lit",)) for b, (s, l) in enumerate(blocks)]
    good = build_container(total, recs)
    i = oracle.info(good)
    bad = good.copy(); bad[64 + (i.n_blocks + 1) * 8 + 5 * 4] ^= 1        # block 0, LIT, lane 5
    expect_corrupt(binding, bad, total, 0)
    bad = good.copy(); bad[i.payload_off + 33] = 1                        # block 0: the LIT word sits at record offset 32
    expect_corrupt(binding, bad, total, 0)
    bad = good.copy(); bad[i.payload_off + 8] = 2                         # n_words[LIT] != 1
    assert open_rc(binding, bad) == binding.E_CORRUPT


# ------------------------------------------------------------------ seeded fuzz over sizes and encoder policies

def test_fuzz_small_containers(binding):
    """120 seeded combinations of profile, size (ragged tails included), offset width, match threshold, depth
    bound, window, in-block level cap and RAW slack; decode_all and every block in isolation, few slots."""
    rng = np.random.default_rng(0xACEA9E)
    kinds = ["markov", "fastq", "genome", "text", "random", "mixed"]
    for it in range(120):
        kind = kinds[it % len(kinds)]
        n = int(rng.integers(1, 14 * B))
        data = W.generate(kind, n, 1000 + it)
        window = int(rng.choice([0, 0, 1, 2, 5]))
        params = dict(min_match=int(rng.choice([4, 5, 8, 16])), max_depth=int(rng.choice([0, 1, 3, 8])), window=window,
                      batch=int(rng.choice([1, 2, 4])) if window else 64, max_level=int(rng.choice([1, 2, 15])),
                      raw_slack_pct=int(rng.choice([0, 0, 25, 1000, 0xFFFFFFFF])), offset_width=int(rng.choice([4, 8])))
        c = oracle.encode(data, **params)
        want = oracle.decode_all(c)
        assert np.array_equal(want, data), (it, kind, n, params)
        full_check(binding, c, want, n_slots=int(rng.choice([1, 3, 64])), n_targets=int(rng.choice([1, 2, 16])))


def test_fuzz_corrupted_containers_never_escape_their_buffers(binding):
    """100 seeded containers with 1-3 flipped bytes anywhere behind the container header: open either rejects
    them or decode_all / decode_blocks run to completion, never write beyond total_len (resp. the listed blocks)
    and report either OK or CORRUPT (a flip inside literal or offset data is not detectable without a checksum)."""
    rng = np.random.default_rng(7)
    seen = {"rejected": 0, "ok": 0, "corrupt": 0}
    for it in range(100):
        kind = ["fastq", "text", "genome", "mixed"][it % 4]
        n = int(rng.integers(2 * B, 9 * B))
        data = W.generate(kind, n, 500 + it)
        c = oracle.encode(data, min_match=8, max_depth=8, window=int(rng.choice([0, 2])), batch=2,
                          raw_slack_pct=int(rng.choice([0, 1000])))
        bad = c.copy()
        for _ in range(int(rng.integers(1, 4))):
            bad[int(rng.integers(64, bad.size))] ^= int(rng.integers(1, 256))
        try:
            dec = binding.Decoder(bad, n_targets=2, n_slots=int(rng.choice([2, 64])))
        except binding.AceapexError:
            seen["rejected"] += 1
            continue
        with dec:
            out = dev_out(n + 4096)
            dec.decode_all(out)
            rc, _ = dec.device_status(clear=True)
            assert rc in (0, binding.E_CORRUPT)
            assert np.all(out.cpu().numpy()[n:] == 0xA5)
            seen["ok" if rc == 0 else "corrupt"] += 1
            ids = np.array([int(rng.integers(0, (n + B - 1) // B)) for _ in range(2)], np.uint64)
            buf = dev_out(2 * B + 64)
            dec.decode_blocks(ids, buf)
            assert dec.device_status(clear=True)[0] in (0, binding.E_CORRUPT)
            assert np.all(buf.cpu().numpy()[2 * B:] == 0xA5)
    assert seen["corrupt"] >= 40                                     # most flips land in entropy-coded data
