"""Shape checks for the seeded synthetic workloads (BASELINE.json configs; DESIGN.md recipe)."""
import numpy as np

from paper_2606_24531_b200 import workloads as W


def test_deterministic_and_seed_sensitive():
    for kind in W.KINDS:
        a = W.generate(kind, 200_000, 5)
        assert np.array_equal(a, W.generate(kind, 200_000, 5))
        assert not np.array_equal(a, W.generate(kind, 200_000, 6))
        if kind != "mixed":   # the mixed chunk order is a shuffle of the whole chunk list
            assert np.array_equal(a[:70_000], W.generate(kind, 70_000, 5))   # prefix-stable


def test_fastq_record_structure():
    d = W.generate("fastq", 1 << 20, W.SEED_BASE + 2).tobytes()
    recs = d.split(b"\n")
    n_full = (len(recs) - 1) // 4
    assert n_full > 3000
    quals = []
    for r in range(0, 200):
        h, seq, plus, q = recs[4 * r: 4 * r + 4]
        assert h == b"@SYN.%d" % (r + 1) and plus == b"+"
        assert len(seq) == 150 and set(seq) <= set(b"ACGTN") and len(q) == 150
        assert all(33 + 2 <= c <= 33 + 41 for c in q)
        quals.append(np.frombuffer(q, np.uint8).astype(float) - 33)
    q = np.mean(quals, axis=0)
    assert 35 < q[:10].mean() < 40 and 23 < q[-10:].mean() < 28       # mean decays 38 -> 25
    bases = b"".join(recs[4 * r + 1] for r in range(n_full))
    assert 0.0005 < bases.count(b"N") / len(bases) < 0.002             # ~0.1% N among bases


def test_genome_alphabet_and_repetition():
    d = W.generate("genome", 4 << 20, W.SEED_BASE + 3)
    assert set(np.unique(d)) == set(b"ACGT")
    cnt = np.bincount(d, minlength=256)[list(b"ACGT")] / d.size
    assert np.all(np.abs(cnt - 0.25) < 0.01)


def test_text_shape():
    d = W.generate("text", 2 << 20, W.SEED_BASE + 4).tobytes()
    lines = d.split(b"\n")
    lens = [len(x) for x in lines[:-1]]
    assert 78 <= np.mean(lens) <= 95 and max(lens) < 100
    words = d.replace(b"\n", b" ").replace(b".", b"").split()
    assert all(2 <= len(w) <= 12 and w.islower() for w in words[:5000])
    sent = [len(s.split()) for s in d.replace(b"\n", b" ").split(b".")[1:200]]
    assert min(sent) >= 8 and max(sent) <= 25
    # Zipf: the most frequent word is much more frequent than the 100th
    from collections import Counter
    c = Counter(words).most_common(100)
    assert c[0][1] > 20 * c[99][1]


def test_markov_alphabet():
    d = W.generate("markov", 1 << 20, W.SEED_BASE + 1)
    assert len(np.unique(d)) <= 64 and d.max() < 128


def test_mixed_quarters():
    n = 64 << 16      # 64 chunks of 64 KiB
    d = W.generate("mixed", n, W.SEED_BASE + 5)
    kinds = {"fastq": 0, "genome": 0, "text": 0, "random": 0}
    for c in range(64):
        ch = d[c << 16:(c + 1) << 16]
        u = len(np.unique(ch))
        if u > 200:
            kinds["random"] += 1
        elif u <= 4:
            kinds["genome"] += 1
        elif (ch == ord("@")).sum() > 100:
            kinds["fastq"] += 1
        else:
            kinds["text"] += 1
    assert all(v == 16 for v in kinds.values()), kinds


def test_seek_ids_seeded_uniform():
    ids = W.seek_ids(65536, 100_000, W.SEED_BASE + 0x75)
    assert ids.dtype == np.uint64 and ids.max() < 65536
    assert np.array_equal(ids, W.seek_ids(65536, 100_000, W.SEED_BASE + 0x75))
    hist = np.bincount((ids >> np.uint64(12)).astype(np.int64), minlength=16)
    assert hist.min() > 5500 and hist.max() < 7000
