"""Pins for the oracle codec (FORMAT.md sections 1-5).

What fixes the oracle here: containers assembled by an independent writer (tests/handmade.py)
whose decoded bytes follow from the plain definition of an absolute-offset copy; round-trip
identity against the original bytes; agreement of two independent decoders on every block; the
closed form for N equal bytes; the validator's invariants; the paper's three-phase isolation
check.
"""
import numpy as np
import pytest

import oracle
from paper_2606_24531_b200 import workloads as W

from handmade import B, BLOG, build_container, build_record, container_from_tokens, expand


def handmade_case():
    """3 blocks: doubling matches with length escapes and tags 1..11; a source spanning two blocks;
    a min-length match; a literal-length escape; a block with no literals at all."""
    total = 2 * B + 100
    seqs0 = [(8, 8, 0)] + [(0, 1 << k, 0) for k in range(4, BLOG)]   # 16 + (B - 16) bytes; BLOG - 3 = 11 matches at 16 KiB
    lits0 = b"ABCDEFGH"
    lits1 = b"0123456789" + bytes((i * 7 + 3) & 0xFF for i in range(300)) + b"tail" * ((B - 328) // 4) + b"xy"
    seqs1 = [(10, 12, B - 5), (300, 4, 3)]
    assert 10 + 12 + 300 + 4 + (len(lits1) - 310) == B
    seqs2 = [(0, 100, B + 10)]
    lits2 = b""
    blocks = [(seqs0, lits0), (seqs1, lits1), (seqs2, lits2)]
    return total, blocks


def test_handmade_container_decodes_to_plain_definition():
    total, blocks = handmade_case()
    want = expand(total, blocks)
    assert want[:16] == b"ABCDEFGHABCDEFGH" and want[B - 5:B] == b"DEFGH"
    assert want[B + 10:B + 22] == b"DEFGH0123456"          # the spanning copy
    c = container_from_tokens(total, blocks)
    assert oracle.decode_all(c).tobytes() == want
    with oracle.Isolated(c) as iso:
        for b in range(3):
            blk, hops = iso.decode(b, with_hops=True)
            assert blk.tobytes() == want[b * B:(b + 1) * B]
        # last byte of block 0 was produced by the 11th match: 11 hops back to a literal
        assert iso.decode(0, with_hops=True)[1] == BLOG - 3
    ll, ml, src, tags = oracle.decode_tokens(c, 0)
    assert list(tags) == list(range(1, BLOG - 2)) and int(ml[-1]) == B // 2
    assert list(oracle.decode_tokens(c, 1)[3]) == [1, 0] and list(oracle.decode_tokens(c, 2)[3]) == [0]
    rep = oracle.validate(c)
    assert rep.n_matches_spanning == 1 and rep.max_level_seen == BLOG - 3 and rep.min_match_seen == 4
    h, lit, ln, off, ex, tg = oracle.decode_streams(c, 1)
    assert h.n_seq == 2 and h.n_extras == 1 and int(ex[0]) == 300 and list(ln) == [10, 8, 255, 0]
    assert h.off_nbytes == 2 and list(off) == [(B - 5) & 255, (B - 5) >> 8, 3, 0]


ADVERSARIAL = {
    "empty": b"",
    "one": b"x",
    "three": b"abc",
    "b_minus_1": bytes((i * 131 + (i >> 5)) & 0xFF for i in range(B - 1)),
    "b_exact": bytes((i * 29 + (i >> 7)) & 0xFF for i in range(B)),
    "b_plus_1": bytes((i * 17 + (i >> 3)) & 0xFF for i in range(B + 1)),
    "all_equal": b"\x00" * (3 * B + 77),
    "all_distinct_cycle": bytes(range(256)) * 200,
    "period2": b"ab" * 30000,
    "period3": b"abc" * 20000,
    "period5": b"abcde" * 15000,
    "two_blocks_text": (b"the quick brown fox jumps over the lazy dog. " * 800)[: 2 * B],
}


@pytest.mark.parametrize("name", sorted(ADVERSARIAL))
@pytest.mark.parametrize("policy", ["literal", "scheduled_small"])
def test_round_trip_adversarial(name, policy):
    data = ADVERSARIAL[name]
    params = dict(min_match=4) if policy == "literal" else dict(min_match=8, max_depth=3, window=2, batch=2, threads=3)
    c = oracle.encode(data, **params)
    assert oracle.decode_all(c).tobytes() == data
    assert oracle.decode_all_mt(c, 4).tobytes() == data
    i = oracle.info(c)
    assert i.total_len == len(data) and i.n_blocks == (len(data) + B - 1) // B
    assert i.container_bytes == c.size
    rep = oracle.validate(c)
    if policy != "literal":
        assert rep.max_depth_seen <= 3
    with oracle.Isolated(c) as iso:
        for b in range(i.n_blocks):
            assert iso.decode(b).tobytes() == data[b * B:(b + 1) * B]


def test_closed_form_equal_bytes_doubling():
    """N equal bytes, T = 4, unbounded chain: 4 literals then matches of 4, 8, 16, ... from
    position 0, the last one cut at the block end (newest source that still fits); tags 1, 2, ..."""
    for n in (4, 7, 8, 9, 100, 4096, B - 3, B):
        c = oracle.encode(b"\x07" * n, min_match=4, chain_depth=1 << 20)
        ll, ml, src, tags = oracle.decode_tokens(c, 0)
        want, want_src, pos = [], [], 4
        while n - pos >= 4:
            m = min(pos, n - pos)
            want.append(m)
            want_src.append(pos - m)   # newest candidate that reaches the limit: 0 while doubling
            pos += m
        assert list(ml) == want and [int(s) for s in src] == want_src
        assert int(ll[0]) == 4 if want else len(ll) == 0
        assert list(tags) == list(range(1, len(want) + 1))
        assert oracle.decode_all(c).tobytes() == b"\x07" * n


def test_zero_match_block_is_order0_coding():
    rng = np.random.default_rng(5)
    data = rng.choice(np.frombuffer(b"ACGT", np.uint8), size=B, p=[0.4, 0.3, 0.2, 0.1]).tobytes()
    c, st = oracle.encode(data, return_stats=True, min_match=B)   # threshold never met: literals only
    assert st.n_seq == 0 and st.n_lit == B
    h = -sum(p * np.log2(p) for p in (0.4, 0.3, 0.2, 0.1)) * B / 8
    payload = c.size - oracle.info(c).payload_off
    assert h * 0.97 <= payload <= h * 1.03 + 32 + 48 + 16 * 8
    assert oracle.decode_all(c).tobytes() == data


def test_uniform_random_ratio_near_one():
    data = W.generate("random", 8 * B, 99)
    c = oracle.encode(data, min_match=4)
    assert 0.93 <= data.size / c.size <= 1.0


PROFILE_SAMPLES = [("markov_1m", 1 << 20), ("fastq_64m", 2 << 20), ("genome_256m", 2 << 20),
                   ("text_256m", 2 << 20), ("mixed_1g", 2 << 20)]


@pytest.mark.parametrize("name,nbytes", PROFILE_SAMPLES)
@pytest.mark.parametrize("policy", ["config", "literal"])
def test_profiles_round_trip_and_decoders_agree(name, nbytes, policy):
    cfg = W.CONFIGS[name]
    data = cfg.data(nbytes)
    params = dict(cfg.encoder) if policy == "config" else dict(W.POLICY_LITERAL)
    if params.get("window"):
        params["window"] = 16           # scaled with the sample so that cross-block matches exist
        params["batch"] = 8
    if name == "markov_1m" and policy == "literal":
        pytest.skip("identical to the config policy")
    c = oracle.encode(data, offset_width=cfg.offset_width, threads=4, **params)
    full = oracle.decode_all(c)
    assert np.array_equal(full, data)
    assert oracle.fnv1a64(full) == oracle.fnv1a64(data)            # PAPER.md:41 FNV check
    for threads in (1, 3):                                           # multi-core driver of the same decoder
        assert np.array_equal(oracle.decode_all_mt(c, threads), data)
    rep = oracle.validate(c)                                         # src+len<=dst, tags, D, R
    assert rep.n_matches_cross + rep.n_matches_intra + rep.n_matches_spanning == rep.n_seq
    if params.get("max_depth"):
        assert rep.max_depth_seen <= params["max_depth"]
    nb = oracle.info(c).n_blocks
    with oracle.Isolated(c) as iso:
        step = 1 if nb <= 64 else 5
        for b in list(range(0, nb, step)) + [nb - 1]:
            assert np.array_equal(iso.decode(b), data[b * B:(b + 1) * B]), b


def test_encoder_result_independent_of_thread_count():
    data = W.generate("text", 1 << 20, 1234)
    a = oracle.encode(data, min_match=8, max_depth=4, window=8, batch=4, threads=1)
    b = oracle.encode(data, min_match=8, max_depth=4, window=8, batch=4, threads=7)
    assert np.array_equal(a, b)


def test_three_phase_isolation_on_the_oracle():
    """PAPER.md:49-51 applied to decoder #2: region differs before, equals after, rest untouched."""
    data = W.generate("fastq", 6 * B, 42)
    c = oracle.encode(data, min_match=8, max_depth=8, window=2, batch=2)
    for fill in (0x00, 0xA5):
        buf = np.full(6 * B, fill, np.uint8)
        target = 4
        region = slice(target * B, (target + 1) * B)
        assert oracle.fnv1a64(buf[region]) != oracle.fnv1a64(data[region])          # phase 1
        with oracle.Isolated(c) as iso:
            buf[region] = iso.decode(target)
        assert oracle.fnv1a64(buf[region]) == oracle.fnv1a64(data[region])          # phase 2
        mask = np.ones(6 * B, bool); mask[region] = False
        assert np.all(buf[mask] == fill)                                             # phase 3


# ---------------------------------------------------------------- invalid containers

def test_rejects_bad_header_fields():
    c = oracle.encode(b"hello hello hello hello")
    for off, val in ((0, ord("X")), (8, 2), (12, 15), (13, 5), (14, 16), (15, 11)):
        bad = c.copy(); bad[off] = val
        with pytest.raises(oracle.OracleError):
            oracle.decode_all(bad)
    with pytest.raises(oracle.OracleError):
        oracle.decode_all(c[:40])
    with pytest.raises(oracle.OracleError):
        oracle.decode_all(c[:-16])


def test_rejects_overlapping_or_forward_match():
    lits = b"abcdefgh" + b"z" * (B - 16)
    for src, ml in ((4, 8), (8, 8), (1 << 20, 8)):      # overlaps dst / starts at dst / beyond
        rec = build_record(0, [(8, ml, src)], lits, tags=[1])
        c = build_container(B, [rec])
        with pytest.raises(oracle.OracleError) as e:
            oracle.decode_all(c)
        assert e.value.code == -4
        with pytest.raises(oracle.OracleError):
            oracle.Isolated(c).decode(0)
        with pytest.raises(oracle.OracleError):
            oracle.validate(c)


def test_rejects_bad_frequency_sum_and_length_mismatch():
    total, blocks = handmade_case()
    good = container_from_tokens(total, blocks)
    i = oracle.info(good)
    bad = good.copy()
    # first u16 frequency of block 0's LIT table: record header 32 B, bitmap 32 B
    p = i.payload_off + 32 + 32
    bad[p] ^= 1
    with pytest.raises(oracle.OracleError):
        oracle.decode_all(bad)
    with pytest.raises(oracle.OracleError):
        oracle.decode_all_mt(bad, 3)
    # block whose tokens do not add up to the block length
    rec = build_record(0, [(8, 8, 0)], b"ABCDEFGH" + b"q" * 10)
    with pytest.raises(oracle.OracleError):
        oracle.decode_all(build_container(B, [rec]))


def test_validator_flags_wrong_tags_and_broken_promises():
    total, blocks = handmade_case()
    recs = [build_record(b * B, s, l) for b, (s, l) in enumerate(blocks)]
    assert oracle.validate(build_container(total, recs)).n_seq == BLOG
    wrong = [build_record(0, blocks[0][0], blocks[0][1], tags=[1] * (BLOG - 3))] + recs[1:]
    with pytest.raises(oracle.OracleError) as e:
        oracle.validate(build_container(total, wrong))
    assert e.value.code == -7
    with pytest.raises(oracle.OracleError) as e:     # depth promise 3 < actual 11
        oracle.validate(build_container(total, recs, max_depth=3))
    assert e.value.code == -7
    with pytest.raises(oracle.OracleError) as e:     # window promise: block 2 reads block 1
        oracle.validate(build_container(total, recs, window=2))
    assert e.value.code == -7


# ---- selective entropy: RAW streams (FORMAT.md section 2 modes)

def test_raw_streams_decode_to_plain_definition():
    """Hand-written records whose streams are stored RAW (no rANS involved at all for the raw ones):
    the decoded bytes are known by construction, for every combination of raw / coded streams."""
    total, blocks = handmade_case()
    want = expand(total, blocks)
    for raw in [("lit",), ("len",), ("off",), ("lit", "len", "off"), ("len", "off")]:
        recs = []
        for b, (seqs, lits) in enumerate(blocks):
            use = tuple(k for k in raw if not (k == "lit" and len(lits) == 0))   # an empty stream cannot be RAW
            recs.append(build_record(b * B, seqs, lits, raw=use))
        c = build_container(total, recs)
        assert oracle.decode_all(c).tobytes() == want, raw
        with oracle.Isolated(c) as iso:
            for b in range(3):
                assert iso.decode(b).tobytes() == want[b * B:(b + 1) * B]
        assert oracle.validate(c).n_matches_spanning == 1
        h, lit, ln, off, ex, tg = oracle.decode_streams(c, 1)
        assert list(ln) == [10, 8, 255, 0] and lit.tobytes() == blocks[1][1]


def test_encoder_picks_raw_only_where_rans_does_not_pay():
    rnd = W.generate("random", 4 * B, 7)
    c, st = oracle.encode(rnd, return_stats=True, min_match=B)            # literals only
    assert list(st.n_raw) == [4, 0, 0]                                   # every LIT stream raw, nothing else exists
    # a raw literal-only block costs its bytes plus index entry, record header and padding
    assert c.size - rnd.size <= 64 + 16 + 4 * (392 + 32 + 16) + 8 + 16
    assert oracle.decode_all(c).tobytes() == rnd.tobytes()
    c0, st0 = oracle.encode(rnd, return_stats=True, min_match=B, raw_slack_pct=0xFFFFFFFF)
    assert list(st0.n_raw) == [0, 0, 0] and c0.size > c.size              # rANS on uniform bytes only adds its table
    assert oracle.decode_all(c0).tobytes() == rnd.tobytes()
    txt = W.generate("text", 4 * B, 7)
    c1, st1 = oracle.encode(txt, return_stats=True, min_match=B)
    assert st1.n_raw[0] == 0                                             # compressible literals stay entropy coded
    # slack widens the margin monotonically and never changes the decoded bytes
    fq = W.generate("fastq", 8 * B, 3)
    prev = None
    for pct in (0, 20, 1000):
        c2, st2 = oracle.encode(fq, return_stats=True, raw_slack_pct=pct)
        assert oracle.decode_all(c2).tobytes() == fq.tobytes()
        n = sum(st2.n_raw)
        assert prev is None or n >= prev
        prev = n
    assert prev == 3 * 8 - (8 - int(np.count_nonzero([oracle.decode_streams(c2, b)[0].n_seq for b in range(8)]))) * 2


def test_rejects_inconsistent_raw_streams():
    total, blocks = handmade_case()
    recs = [build_record(b * B, s, l, raw=("len",)) for b, (s, l) in enumerate(blocks)]
    good = build_container(total, recs)
    assert oracle.decode_all(good).tobytes() == expand(total, blocks)
    i = oracle.info(good)

    def rejected(c):
        with pytest.raises(oracle.OracleError):
            oracle.decode_all(c)

    bad = good.copy(); bad[i.payload_off + 7] = 0x0C                      # reserved mode 3 for LEN
    rejected(bad)
    bad = good.copy(); bad[i.payload_off + 7] |= 0x40                     # reserved bits 6-7
    rejected(bad)
    bad = good.copy(); bad[i.payload_off + 8 + 4] ^= 1                    # n_words[LEN] != ceil(n_sym / 2)
    rejected(bad)
    bad = good.copy()
    st = 64 + (i.n_blocks + 1) * 8 + (0 * 3 + 1) * 32 * 4 + 7 * 4         # block 0, LEN stream, lane 7
    bad[st] ^= 1                                                          # an unused state that is not 2^16
    rejected(bad)
    # pad byte of an odd-length raw stream must be zero: block 2 has 1 sequence -> OFF stream of 2 bytes (even),
    # so use a 3-byte literal stream
    rec, stt = build_record(0, [], b"abc", raw=("lit",))
    c = build_container(3, [(rec, stt)])
    assert oracle.decode_all(c).tobytes() == b"abc"
    pos = oracle.info(c).payload_off + 32 + 3                             # first section after the header = words[LIT]
    bad = c.copy(); assert bad[pos] == 0; bad[pos] = 1
    rejected(bad)


def test_seek_aware_policy_bounds_fanout_and_depth_and_validator_checks_them():
    """SURVEY.md section 8f rank 4 (a seek needs every block a block copies from): max_fanout F and
    max_depth D are header promises; the validator recomputes both from the tokens alone."""
    cfg = W.CONFIGS["text_256m"]
    data = cfg.data(3 * 1024 * 1024)
    base = dict(W.POLICY_SCHEDULED, window=16, batch=8)                # a window the 192-block sample can use
    c0 = oracle.encode(data, offset_width=4, **base)
    r0 = oracle.validate(c0)
    assert r0.max_src_blocks_per_block > 12                            # the unbounded policy really fans out
    for F, D in ((12, 8), (4, 2)):
        c = oracle.encode(data, offset_width=4, **dict(base, max_fanout=F, max_depth=D))
        assert np.array_equal(oracle.decode_all(c), data)
        i = oracle.info(c)
        assert (i.max_fanout, i.max_depth, i.min_match_policy) == (F, D, 8)
        r = oracle.validate(c)                                         # raises if a promise is broken
        assert r.max_src_blocks_per_block <= F and r.max_depth_seen <= D
        assert c.size >= c0.size                                       # a bound can only cost ratio
    # a container that promises less than it keeps: same tokens, header fan-out lowered to 2
    bad = c0.copy()
    bad[46:48] = np.frombuffer(np.uint16(2).tobytes(), np.uint8)
    assert np.array_equal(oracle.decode_all(bad), data)                # decoding never depends on a promise
    with pytest.raises(oracle.OracleError) as e:
        oracle.validate(bad)
    assert e.value.code == -7


def test_long_hash_finds_longer_matches_and_round_trips():
    """SURVEY.md reading A14: optional 12-byte long hash, probed first. Same format, same decoders."""
    cfg = W.CONFIGS["genome_256m"]
    data = cfg.data(2 * 1024 * 1024)
    short = dict(W.POLICY_SCHEDULED, window=16, batch=8)
    c_s, st_s = oracle.encode(data, return_stats=True, offset_width=8, **short)
    c_l, st_l = oracle.encode(data, return_stats=True, offset_width=8, threads=3, **dict(short, long_hash=12))
    c_l1 = oracle.encode(data, offset_width=8, threads=1, **dict(short, long_hash=12))
    assert np.array_equal(c_l, c_l1)                                   # independent of the thread count
    assert np.array_equal(oracle.decode_all(c_l), data)
    oracle.validate(c_l)
    assert st_l.match_bytes / st_l.n_seq > st_s.match_bytes / st_s.n_seq and c_l.size < c_s.size
    with oracle.Isolated(c_l) as iso:
        for b in (0, 57, 127):
            assert np.array_equal(iso.decode(b), data[b * 16384:(b + 1) * 16384])


def test_max_seq_caps_sequences_per_block():
    """Encoder knob max_seq: a block never holds more sequences; what follows in the block is literal."""
    data = W.generate("text", 1 << 20, 99)
    base = dict(min_match=4, chain_depth=32)
    c0, st0 = oracle.encode(data, return_stats=True, **base)
    c1, st1 = oracle.encode(data, return_stats=True, max_seq=300, **base)
    assert np.array_equal(oracle.decode_all(c1), data)
    oracle.validate(c1)
    n0 = [oracle.decode_streams(c0, b)[0].n_seq for b in range(64)]
    n1 = [oracle.decode_streams(c1, b)[0].n_seq for b in range(64)]
    assert max(n0) > 300 and max(n1) == 300 and st1.n_seq < st0.n_seq and c1.size > c0.size


# ---- selective entropy: CONST streams (FORMAT.md section 2 mode 2; SURVEY.md section 8f rank 1 "RAW / CONST / rANS")

def const_case():
    """2 blocks whose streams are constant by construction: block 0 is B equal literals (LIT constant, no sequences);
    block 1 repeats the sequence (5 literals 'y', a 9-byte copy of out[7..16)) so that LIT, LEN (5, 5) and OFF (7, one
    byte) are all constant streams."""
    k = B // 14
    blocks = [([], b"q" * B), ([(5, 9, 7)] * k, b"y" * (5 * k + (B - 14 * k)))]
    return 2 * B, blocks


def test_const_streams_decode_to_plain_definition():
    total, blocks = const_case()
    want = expand(total, blocks)
    assert want[:B] == b"q" * B and want[B:B + 14] == b"yyyyy" + b"q" * 9
    for const in [("lit",), ("len",), ("off",), ("lit", "len", "off")]:
        recs = []
        for b, (seqs, lits) in enumerate(blocks):
            use = tuple(k for k in const if k == "lit" or seqs)           # block 0 has no LEN / OFF symbols at all
            recs.append(build_record(b * B, seqs, lits, const=use))
        c = build_container(total, recs)
        assert oracle.decode_all(c).tobytes() == want, const
        with oracle.Isolated(c) as iso:
            for b in range(2):
                assert iso.decode(b).tobytes() == want[b * B:(b + 1) * B]
        oracle.validate(c)
        h, lit, ln, off, ex, tg = oracle.decode_streams(c, 1)
        assert set(ln) == {5} and set(off) == {7} and h.off_nbytes == 1 and set(lit) == {ord("y")}
    # a constant stream costs one word instead of a 34-byte table
    plain = build_container(total, [build_record(b * B, s, l) for b, (s, l) in enumerate(blocks)])
    assert c.size < plain.size


def test_encoder_stores_one_symbol_streams_as_const():
    data = ADVERSARIAL["all_equal"]                                        # 3 blocks + 77 equal bytes
    c, st = oracle.encode(data, return_stats=True)
    assert np.array_equal(oracle.decode_all(c), np.frombuffer(data, np.uint8))
    assert st.n_const[oracle.LIT] == 1 and sum(st.n_const) == 1            # block 0's four equal literals
    c0, st0 = oracle.encode(data, return_stats=True, raw_slack_pct=0xFFFFFFFF)   # selective entropy off: rANS everywhere
    assert sum(st0.n_const) == 0 and sum(st0.n_raw) == 0 and c.size < c0.size
    assert np.array_equal(oracle.decode_all(c0), oracle.decode_all(c))
    with oracle.Isolated(c) as iso:
        for b in range(4):
            assert iso.decode(b).tobytes() == data[b * B:(b + 1) * B]


def test_rejects_inconsistent_const_streams():
    total, blocks = const_case()
    recs = [build_record(b * B, s, l, const=("lit",)) for b, (s, l) in enumerate(blocks)]
    good = build_container(total, recs)
    assert oracle.decode_all(good).tobytes() == expand(total, blocks)
    i = oracle.info(good)

    def rejected(c):
        with pytest.raises(oracle.OracleError):
            oracle.decode_all(c)

    bad = good.copy(); bad[i.payload_off + 8] = 2                         # n_words[LIT] != 1
    rejected(bad)
    bad = good.copy(); bad[i.payload_off + 7] = 0x03                      # reserved mode 3 for LIT
    rejected(bad)
    bad = good.copy(); bad[i.payload_off + 20] = 34                       # a table section beside a CONST stream
    rejected(bad)
    bad = good.copy(); bad[64 + (i.n_blocks + 1) * 8 + 5 * 4] ^= 1        # block 0, LIT, lane 5: a state that is not 2^16
    rejected(bad)
    # block 0's record: header 32 bytes, no tables, no extras, no tags -> the LIT word sits at offset 32
    assert good[i.payload_off + 32] == ord("q")
    bad = good.copy(); bad[i.payload_off + 33] = 1                        # high byte of the word must be zero
    rejected(bad)
