"""Pins for the oracle's entropy layer (FORMAT.md section 3; PAPER.md:33, :124 ref [6]).

None of these re-types the oracle's formula: they compare against hand-worked values
(tests/golden/rans_worked_values.txt), closed forms, brute-force round trips,
the information identity and the end-state invariant.
"""
import itertools
import math

import numpy as np
import pytest

import oracle

A, Bsym = ord("a"), ord("b")


def table_ab():
    f = np.zeros(256, np.uint16)
    f[A], f[Bsym] = 4000, 96
    return f


def ints(s):
    return [int(x, 0) for x in s.split()]


def test_worked_case_i(golden_rans):
    st, w = oracle.rans_encode(b"b", table_ab())
    assert len(w) == int(golden_rans["case_i.n_words"])
    assert int(st[0]) == int(golden_rans["case_i.state0"], 0)
    assert all(int(x) == 65536 for x in st[1:])
    # the decoder alone, fed the hand-worked state, must give "b" and end at 2^16
    init = np.full(32, 65536, np.uint32)
    init[0] = int(golden_rans["case_i.state0"], 0)
    assert oracle.rans_decode(init, np.zeros(0, np.uint16), table_ab(), 1).tobytes() == b"b"


def test_worked_case_ii(golden_rans):
    st, w = oracle.rans_encode(b"b" * 96, table_ab())
    assert len(w) == int(golden_rans["case_ii.n_words"])
    assert all(int(x) == int(golden_rans["case_ii.word_all"], 0) for x in w)
    assert all(int(x) == int(golden_rans["case_ii.state_all"], 0) for x in st)
    # the trace itself, by plain arithmetic on the golden numbers: x -> (x//f << 12) + x%f + c
    tr = ints(golden_rans["case_ii.trace"])
    assert tr[1] == ((tr[0] // 96) << 12) + tr[0] % 96 + 4000
    assert tr[2] == ((tr[1] // 96) << 12) + tr[1] % 96 + 4000
    assert tr[2] >= 96 << 20 and (tr[2] & 0xFFFF) == int(golden_rans["case_ii.word_all"], 0)
    x = tr[2] >> 16
    assert tr[3] == ((x // 96) << 12) + x % 96 + 4000
    # decoder alone from golden states/words
    init = np.full(32, int(golden_rans["case_ii.state_all"], 0), np.uint32)
    words = np.full(32, int(golden_rans["case_ii.word_all"], 0), np.uint16)
    assert oracle.rans_decode(init, words, table_ab(), 96).tobytes() == b"b" * 96


def test_worked_case_iii_order_sensitive(golden_rans):
    msg = bytes(Bsym if (i * i + i // 3) % 7 == 3 else A for i in range(4096))
    assert msg.count(b"b") == int(golden_rans["case_iii.count_b"])
    st, w = oracle.rans_encode(msg, table_ab())
    assert len(w) == int(golden_rans["case_iii.n_words"])
    assert [int(x) for x in w[:4]] == ints(golden_rans["case_iii.words_first4"])
    assert int(w[-1]) == int(golden_rans["case_iii.word_last"], 0)
    assert [int(x) for x in st[:4]] == ints(golden_rans["case_iii.states_0_3"])
    assert int(st[31]) == int(golden_rans["case_iii.state_31"], 0)
    assert oracle.fnv1a64(w.astype("<u2").tobytes()) == int(golden_rans["case_iii.fnv_words_le"], 0)
    assert oracle.fnv1a64(st.astype("<u4").tobytes()) == int(golden_rans["case_iii.fnv_states_le"], 0)
    assert oracle.rans_decode(st, w, table_ab(), 4096).tobytes() == msg


def test_fnv_standard_vectors(golden_rans):
    assert oracle.fnv1a64(b"") == int(golden_rans["fnv.empty"], 0)
    assert oracle.fnv1a64(b"a") == int(golden_rans["fnv.a"], 0)
    assert oracle.fnv1a64(b"foobar") == 0x85944171F73967E8  # published FNV-1a-64 test vector


def test_information_identity(golden_rans):
    """16*n_words + sum log2(x_l / 2^16) ~= sum log2(4096 / f[s_i])."""
    msg = bytes(Bsym if i % 5 == 0 else A for i in range(200))
    f = table_ab()
    st, w = oracle.rans_encode(msg, f)
    coded = 16 * len(w) + sum(math.log2(int(x) / 65536.0) for x in st)
    info = sum(math.log2(4096.0 / int(f[c])) for c in msg)
    assert len(w) == int(golden_rans["info_identity.n_words"])
    assert abs(coded - float(golden_rans["info_identity.coded_bits"])) < 0.01
    assert abs(info - float(golden_rans["info_identity.info_bits"])) < 0.01
    # general form on a longer skewed message: rANS loses < 0.01 bit/symbol + O(1) per lane
    rng = np.random.default_rng(7)
    cnt = np.zeros(256, np.uint32)
    sym = rng.choice(np.arange(40, 60), size=20000, p=np.arange(1, 21) / 210.0).astype(np.uint8)
    for s in sym:
        cnt[s] += 1
    fq = oracle.quantise(cnt)
    st, w = oracle.rans_encode(sym, fq)
    coded = 16 * len(w) + sum(math.log2(int(x) / 65536.0) for x in st)
    info = sum(math.log2(4096.0 / int(fq[s])) for s in sym)
    assert info - 1e-6 <= coded + 32 * 1e-3 and coded - info < 0.01 * len(sym) + 32


@pytest.mark.parametrize("lanes", [1, 32])
@pytest.mark.parametrize("split", [(4095, 1), (2048, 2048), (4000, 96), (1, 4095)])
def test_bruteforce_two_symbols(lanes, split):
    """every string of length <= 11 over {a,b}: decode(encode(s)) == s, end states == 2^16 (checked
    inside ora_rans_decode), exact word count consumed."""
    f = np.zeros(256, np.uint16)
    f[A], f[Bsym] = split
    for n in range(0, 12):
        for tup in itertools.product((A, Bsym), repeat=n):
            s = bytes(tup)
            st, w = oracle.rans_encode(s, f, lanes=lanes)
            assert oracle.rans_decode(st, w, f, n, lanes=lanes).tobytes() == s


@pytest.mark.parametrize("lanes", [1, 32])
@pytest.mark.parametrize("split", [(4094, 1, 1), (1366, 1365, 1365), (1, 2, 4093)])
def test_bruteforce_three_symbols(lanes, split):
    f = np.zeros(256, np.uint16)
    f[0], f[7], f[255] = split
    for n in range(0, 8):
        for tup in itertools.product((0, 7, 255), repeat=n):
            s = bytes(tup)
            st, w = oracle.rans_encode(s, f, lanes=lanes)
            assert oracle.rans_decode(st, w, f, n, lanes=lanes).tobytes() == s


def test_long_low_probability_runs_renormalise_once_per_symbol():
    """f = 1 symbols force a word on almost every step; one step must suffice (FORMAT.md 3)."""
    f = np.zeros(256, np.uint16)
    f[0], f[1] = 4095, 1
    s = bytes([1]) * 5000 + bytes([0]) * 100 + bytes([1]) * 333
    for lanes in (1, 5, 32):
        st, w = oracle.rans_encode(s, f, lanes=lanes)
        assert len(w) <= len(s)
        assert oracle.rans_decode(st, w, f, len(s), lanes=lanes).tobytes() == s
        assert all(65536 <= int(x) < 2 ** 32 for x in st)


def test_decoder_rejects_wrong_word_count_and_bad_end_state():
    f = table_ab()
    msg = bytes(Bsym if i % 3 == 0 else A for i in range(1000))
    st, w = oracle.rans_encode(msg, f)
    with pytest.raises(oracle.OracleError):
        oracle.rans_decode(st, np.concatenate([w, np.zeros(1, np.uint16)]), f, len(msg))
    with pytest.raises(oracle.OracleError):
        oracle.rans_decode(st, w[:-1], f, len(msg))
    bad = st.copy()
    bad[3] ^= 0x10000
    with pytest.raises(oracle.OracleError):
        oracle.rans_decode(bad, w, f, len(msg))


def test_single_symbol_stream_costs_nothing():
    f = np.zeros(256, np.uint16)
    f[65] = 4096
    st, w = oracle.rans_encode(b"A" * 10000, f)
    assert len(w) == 0 and all(int(x) == 65536 for x in st)
    assert oracle.rans_decode(st, w, f, 10000).tobytes() == b"A" * 10000


def test_quantiser_properties():
    rng = np.random.default_rng(3)
    for trial in range(200):
        k = int(rng.integers(1, 257))
        cnt = np.zeros(256, np.uint32)
        idx = rng.choice(256, size=k, replace=False)
        cnt[idx] = rng.integers(1, 1 + int(rng.choice([2, 50, 100000])), size=k)
        f = oracle.quantise(cnt)
        assert int(f.astype(np.int64).sum()) == 4096
        assert np.all((f > 0) == (cnt > 0))
    # closed forms: one symbol -> 4096; two equal counts -> 2048/2048; 4095:1 -> exact
    c = np.zeros(256, np.uint32); c[9] = 5
    assert int(oracle.quantise(c)[9]) == 4096
    c = np.zeros(256, np.uint32); c[1] = c[2] = 77
    assert [int(x) for x in oracle.quantise(c)[1:3]] == [2048, 2048]
    c = np.zeros(256, np.uint32); c[0] = 4095; c[200] = 1
    q = oracle.quantise(c)
    assert int(q[0]) == 4095 and int(q[200]) == 1
    # remainder goes to the largest count, ties to the lower symbol
    c = np.zeros(256, np.uint32); c[10] = c[20] = c[30] = 1
    q = oracle.quantise(c)
    assert [int(q[10]), int(q[20]), int(q[30])] == [1366, 1365, 1365]
    assert not oracle.quantise(np.zeros(256, np.uint32)).any()


def test_uniform_random_bytes_do_not_compress():
    rng = np.random.default_rng(11)
    s = rng.integers(0, 256, size=16384, dtype=np.uint8)
    cnt = np.bincount(s, minlength=256).astype(np.uint32)
    f = oracle.quantise(cnt)
    st, w = oracle.rans_encode(s, f)
    coded_bytes = 2 * len(w) + 4 * 32
    h0 = -sum((c / 16384.0) * math.log2(c / 16384.0) for c in cnt if c) * 16384 / 8
    assert h0 - 8 <= coded_bytes <= 1.02 * 16384 + 128
