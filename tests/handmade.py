"""A second, independent container *writer* used only by tests.

It lays out the header, the index and the block records of FORMAT.md sections 1-2 and the token
grammar of section 4 in plain Python from explicit token lists, so that tests can (a) pin the
oracle decoders on containers whose decoded bytes are known by construction and (b) feed the
CUDA path streams the oracle encoder never produces (sources that span two blocks, length
escapes, deep tag chains, corrupt fields). Only the per-stream rANS coding is borrowed from the
oracle (`oracle.rans_encode`, itself pinned by tests/test_oracle_rans.py).
"""
from __future__ import annotations

import os
import struct

import numpy as np

import oracle

# Block size: 16 KiB unless ACEAPEX_BLOCK_LOG2 selects another one (block-size sweep: the oracle pins are
# re-run against the variant, tests/test_oracle_blocksize.py).
BLOG = int(os.environ.get("ACEAPEX_BLOCK_LOG2", "14"))
B = 1 << BLOG


def pad16(n):
    return (n + 15) & ~15


def _table(freq):
    bitmap = bytearray(32)
    body = b""
    for s in range(256):
        if freq[s]:
            bitmap[s >> 3] |= 1 << (s & 7)
            body += struct.pack("<H", int(freq[s]))
    return bytes(bitmap) + body


def _stream(sym: bytes, freq=None):
    """-> (table bytes, words bytes, n_words, states[32])"""
    if len(sym) == 0:
        return b"", b"", 0, [65536] * 32
    if freq is None:
        freq = oracle.quantise(np.bincount(np.frombuffer(sym, np.uint8), minlength=256).astype(np.uint32))
    st, w = oracle.rans_encode(sym, freq)
    return _table(freq), w.astype("<u2").tobytes(), len(w), [int(x) for x in st]


def compute_tags(block_start, seqs):
    """FORMAT.md section 4 'tags', recomputed from (lit_len, match_len, src) triples."""
    level = np.zeros(B, np.int32)
    pos = block_start
    tags = []
    for ll, ml, src in seqs:
        pos += ll
        lv = 0
        for p in range(max(src, block_start), src + ml):
            lv = max(lv, int(level[p - block_start]) + 1)
        tags.append(lv)
        level[pos - block_start: pos - block_start + ml] = lv
        pos += ml
    return tags


def _raw_stream(sym: bytes):
    """FORMAT.md section 2, mode 1 (RAW): no table, the symbols verbatim in the words section."""
    assert len(sym) >= 1
    body = bytes(sym) + (b"\0" if len(sym) & 1 else b"")
    return b"", body, len(body) // 2, [65536] * 32


def _const_stream(sym: bytes):
    """FORMAT.md section 2, mode 2 (CONST): no table, one word whose low byte is the repeated symbol."""
    assert len(sym) >= 1 and len(set(sym)) == 1
    return b"", bytes([sym[0], 0]), 1, [65536] * 32


def build_record(block_start, seqs, literals: bytes, off_width=4, tags=None, off_nbytes=None, freqs=None, raw=(), const=()):
    """seqs: list of (lit_len, match_len, src). `literals`: all literal bytes of the block.
    raw: names of the streams ("lit", "len", "off") to store RAW instead of rANS-coded."""
    if tags is None:
        tags = compute_tags(block_start, seqs)
    if off_nbytes is None:
        m = max([s[2] for s in seqs], default=0)
        off_nbytes = 1
        while off_nbytes < 8 and (m >> (8 * off_nbytes)):
            off_nbytes += 1
    assert off_nbytes <= off_width
    len_sym, off_sym, extras = bytearray(), bytearray(), []
    for ll, ml, src in seqs:
        len_sym.append(min(ll, 255))
        if ll >= 255:
            extras.append(ll)
        len_sym.append(min(ml - 4, 255))
        if ml - 4 >= 255:
            extras.append(ml - 4)
        off_sym += int(src).to_bytes(8, "little")[:off_nbytes]
    freqs = freqs or {}
    syms = {"lit": bytes(literals), "len": bytes(len_sym), "off": bytes(off_sym)}
    streams = [_raw_stream(syms[k]) if k in raw else (_const_stream(syms[k]) if k in const else _stream(syms[k], freqs.get(k)))
               for k in ("lit", "len", "off")]
    modes = sum((1 if k in raw else 2) << (2 * i) for i, k in enumerate(("lit", "len", "off")) if k in raw or k in const)
    hdr = struct.pack("<HHHBB", len(seqs), len(literals), len(extras), off_nbytes, modes)
    hdr += struct.pack("<III", *(s[2] for s in streams))
    hdr += struct.pack("<HHH", *(len(s[0]) for s in streams))
    hdr += b"\0" * 6
    assert len(hdr) == 32
    rec = bytearray(hdr)

    def section(data):
        nonlocal rec
        rec += b"\0" * (pad16(len(rec)) - len(rec))
        rec += data

    for s in streams:
        section(s[0])
    section(b"".join(struct.pack("<H", e) for e in extras))
    tagbytes = bytearray((len(seqs) + 1) // 2)
    for k, t in enumerate(tags):
        tagbytes[k >> 1] |= (t & 15) << ((k & 1) * 4)
    section(bytes(tagbytes))
    for s in streams:
        section(s[1])
    rec += b"\0" * (pad16(len(rec)) - len(rec))
    return bytes(rec), [s[3] for s in streams]


def build_container(total_len, records, off_width=4, max_depth=0, window=0, max_level=15, min_match=4,
                    magic=b"ACEAPEX1", version=1):
    """records: list of (record bytes, states[3][32]) per block, in block order."""
    nb = (total_len + B - 1) // B
    assert nb == len(records)
    index_bytes = (nb + 1) * 8 + nb * 3 * 32 * 4
    payload_off = pad16(64 + index_bytes)
    hdr = magic + struct.pack("<IBBBB", version, BLOG, off_width, 32, 12)
    hdr += struct.pack("<QQ", total_len, nb)
    hdr += struct.pack("<IIII", max_depth, window, max_level, min_match)
    hdr += struct.pack("<QQ", 64, payload_off)
    assert len(hdr) == 64
    offs, o = [], 0
    for rec, _ in records:
        offs.append(o)
        o += len(rec)
    offs.append(o)
    idx = b"".join(struct.pack("<Q", x) for x in offs)
    for _, st in records:
        for s in range(3):
            idx += b"".join(struct.pack("<I", x) for x in st[s])
    out = bytearray(hdr + idx)
    out += b"\0" * (payload_off - len(out))
    for rec, _ in records:
        out += rec
    return np.frombuffer(bytes(out), dtype=np.uint8).copy()


def expand(total_len, blocks):
    """Reference expansion of explicit tokens by the plain definition: literals, then
    memcpy from the absolute position. blocks: list of (seqs, literals)."""
    out = bytearray(total_len)
    for b, (seqs, lits) in enumerate(blocks):
        pos, lp = b * B, 0
        for ll, ml, src in seqs:
            out[pos:pos + ll] = lits[lp:lp + ll]
            pos += ll; lp += ll
            assert src + ml <= pos
            out[pos:pos + ml] = out[src:src + ml]
            pos += ml
        rest = len(lits) - lp
        out[pos:pos + rest] = lits[lp:]
        pos += rest
        assert pos == min((b + 1) * B, total_len), (b, pos)
    return bytes(out)


def container_from_tokens(total_len, blocks, **kw):
    off_width = kw.get("off_width", 4)
    recs = [build_record(b * B, seqs, lits, off_width=off_width) for b, (seqs, lits) in enumerate(blocks)]
    return build_container(total_len, recs, **kw)
