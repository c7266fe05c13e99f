// Isolated decode (seek / decode_blocks): per-byte origin chase through the compressed data
// ("a match referencing absolute position p can be resolved as soon as the block
// containing p is available"; only the target block is written). SURVEY.md
// section 8(c) reading A7: the paper does not say where a seeked block gets source bytes that
// live in other blocks; here every needed position is followed, hop by hop, through the token
// streams of the block that owns it until it lands on a literal.
//
// State: pend[i][o] = the absolute position whose byte value equals output byte o of target i
// (initially the byte's own position), or kDone. One hop = collect the distinct blocks the
// pending positions fall in -> entropy-decode + parse those blocks into slots -> resolve: a
// position inside a literal run yields the byte; a position inside match k moves to
// src_k + (o - dst_k), which is strictly smaller (src + len <= dst), so the chase terminates.
#pragma once
#include "match.cuh"

namespace aceapex {

constexpr uint32_t kChunk = 16;   // output bytes per thread in the per-byte kernels

__global__ void k_seek_init(Container cv, const uint64_t *ids, uint32_t n_targets, uint64_t *pend)
{
    const uint64_t g = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;      // one thread per byte
    if (g >= (uint64_t)n_targets * kB) return;
    const uint32_t i = (uint32_t)(g >> kBlockLog2), o = (uint32_t)(g & (kB - 1));
    const uint64_t id = ids[i];
    pend[g] = (id < cv.n_blocks && o < block_len_of(cv, id)) ? (id << kBlockLog2) + o : kDone;
}

// Claim a slot for every distinct block that a pending position falls in.
__global__ void k_seek_collect(const uint64_t *pend, uint64_t n_bytes, uint32_t *mark, uint32_t *slot_of,
                               uint64_t *list, Control *ctl, uint32_t tag, uint32_t max_slots)
{
    const uint64_t c = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const uint64_t g0 = c * kChunk;
    if (g0 >= n_bytes) return;
    uint64_t last = kDone;
    for (uint32_t j = 0; j < kChunk; j++) {
        const uint64_t p = pend[g0 + j];
        if (p == kDone) continue;
        const uint64_t blk = p >> kBlockLog2;
        if (blk == last) continue;
        last = blk;
        if (mark[blk] == tag) continue;
        if (atomicExch(mark + blk, tag) == tag) continue;     // somebody else claimed it
        const uint32_t s = atomicAdd(&ctl->n_list, 1u);
        slot_of[blk] = s;                                      // s >= max_slots: no slot this hop
        if (s < max_slots) list[s] = blk;
    }
}

// Resolve every pending position whose block holds a slot in this hop.
//   out mapping: packed -> target i at out + (out_base + i) * 16384; absolute -> out + ids[i] * 16384.
__global__ void k_seek_resolve(Container cv, SlotLayout sl, const uint8_t *slots, uint64_t *pend,
                               uint32_t n_targets, const uint64_t *ids, const uint32_t *mark,
                               const uint32_t *slot_of, Control *ctl, uint32_t tag, uint32_t max_slots,
                               uint8_t *out, uint64_t out_base, uint32_t absolute)
{
    const uint64_t c = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const uint64_t g0 = c * kChunk;
    uint32_t remaining = 0;
    if (g0 < (uint64_t)n_targets * kB) {
        const uint32_t i = (uint32_t)(g0 >> kBlockLog2);
        uint8_t *dst = out + ((absolute ? ids[i] : out_base + i) << kBlockLog2) + (g0 & (kB - 1));
        // cache of the sequence found for the previous byte
        uint64_t c_blk = kDone;
        const uint8_t *c_slot = nullptr;
        uint32_t c_q = 0, c_lo = 1, c_hi = 0, c_nseq = 0, c_blen = 0;
        const uint16_t *c_start = nullptr;
        for (uint32_t j = 0; j < kChunk; j++) {
            const uint64_t p = pend[g0 + j];
            if (p == kDone) continue;
            const uint64_t blk = p >> kBlockLog2;
            const uint32_t o = (uint32_t)(p & (kB - 1));
            if (blk != c_blk) {
                c_blk = blk;
                c_slot = nullptr;
                c_lo = 1; c_hi = 0;
                if (mark[blk] == tag) {
                    const uint32_t s = slot_of[blk];
                    if (s < max_slots) {
                        c_slot = slots + (size_t)s * sl.stride;
                        const SlotHdr *h = reinterpret_cast<const SlotHdr *>(c_slot + sl.o_hdr);
                        if (!h->parsed_ok) {
                            c_slot = nullptr;
                            c_blk = kDone;
                            pend[g0 + j] = kDone;              // corrupt block: give up on this byte
                            raise(ctl, kStChase, blk);
                            continue;
                        }
                        c_nseq = h->n_seq;
                        c_blen = h->block_len;
                        c_start = reinterpret_cast<const uint16_t *>(c_slot + sl.o_start);
                    }
                }
            }
            if (!c_slot) { remaining++; continue; }            // no slot this hop: try again next hop
            if (o >= c_blen) { pend[g0 + j] = kDone; raise(ctl, kStChase, blk); continue; }
            if (!(o >= c_lo && o < c_hi)) {
                // largest q in [0, n_seq] with start[q] <= o (start[0] == 0)
                uint32_t lo = 0, hi = c_nseq;
                while (lo < hi) {
                    const uint32_t mid = (lo + hi + 1) >> 1;
                    if (c_start[mid] <= o) lo = mid; else hi = mid - 1;
                }
                c_q = lo;
                c_lo = c_start[lo];
                c_hi = lo < c_nseq ? c_start[lo + 1] : c_blen;
            }
            const uint32_t q = c_q;
            const uint32_t d = q < c_nseq ? reinterpret_cast<const uint16_t *>(c_slot + sl.o_dst)[q] : c_blen;
            if (o < d) {                                       // a literal: the origin
                const uint32_t lp = reinterpret_cast<const uint16_t *>(c_slot + sl.o_litpos)[q];
                dst[j] = c_slot[sl.o_lit + lp + (o - c_lo)];
                pend[g0 + j] = kDone;
            } else {                                           // a match: follow the absolute offset
                const uint64_t nxt = reinterpret_cast<const uint64_t *>(c_slot + sl.o_src)[q] + (o - d);
                if (nxt >= p) { pend[g0 + j] = kDone; raise(ctl, kStChase, blk); continue; }
                pend[g0 + j] = nxt;
                remaining++;
            }
        }
    }
    // CTA-level count of what is still pending
    __shared__ uint32_t s_rem;
    if (threadIdx.x == 0) s_rem = 0;
    __syncthreads();
    if (remaining) atomicAdd(&s_rem, remaining);
    __syncthreads();
    if (threadIdx.x == 0 && s_rem) atomicAdd(&ctl->pending, (unsigned long long)s_rem);
}

// After the promised number of hops nothing may be pending (header promise D, FORMAT.md section 1).
__global__ void k_seek_check(Control *ctl)
{
    if (ctl->pending != 0) raise(ctl, kStChase, 0);
}

}  // namespace aceapex
