// Isolated decode (seek / decode_blocks): per-byte origin chase through the compressed data
// ("a match referencing absolute position p can be resolved as soon as the block
// containing p is available"; only the target block is written). SURVEY.md
// section 8(c) reading A7: the paper does not say where a seeked block gets source bytes that
// live in other blocks; here every needed position is followed through the token streams of the
// block that owns it until it lands on a literal.
//
// State: pend[i][o] = the absolute position whose byte value equals output byte o of target i
// (initially the byte's own position), a literal request (slot + index into its LIT stream) once the
// chase has reached a literal, or kDone. A position inside match k moves to src_k + (o - dst_k), which
// is strictly smaller (src + len <= dst), so the chase terminates.
#pragma once
#include <cooperative_groups.h>

#include "match.cuh"

namespace aceapex {

// ---------------------------------------------------------------------------------------------
// Fused isolated decode: the whole hop loop in ONE kernel (north_star: "a fused single-block seek
// path that does entropy decode, then gathers source bytes, then copies"). All CTAs are resident
// (the host sizes the grid from the occupancy query), so the phases of a hop are separated by a
// grid barrier instead of kernel boundaries, and the loop ends on the device when nothing is pending:
// one launch per seek, no host read-back.

// Grid barrier for the co-resident CTAs of the cooperative launch (the runtime's own grid sync: measured 6 %
// faster per seek than a hand-rolled counter + generation barrier with acquire polling).
__device__ inline void grid_barrier()
{
    cooperative_groups::this_grid().sync();
}

// Parse the decoded LEN / OFF streams of the block in `slot` into the slot's token arrays (FORMAT.md
// section 4; same rules as the match kernel's parse). FOUR warps share a block, each a contiguous
// quarter of its sequences (the phase is pure latency, so the rounds are spread): pass 0 counts the
// length escapes of each quarter, pass 1 sums the lengths, pass 2 - with the quarter's bases known -
// scans and writes start / dst / litpos / src and checks every match. The passes are separated by CTA
// barriers: all warps of the CTA call this the same number of times (idle quads pass slot == nullptr).
//   sq: shared exchange area of the quad, uint32_t [4][4].
__device__ inline void quad_parse_block(const Container &cv, const SlotLayout &sl, uint8_t *slot, uint64_t blk,
                                        Control *ctl, uint32_t lane, uint32_t r /* warp in quad */, uint32_t (*sq)[4])
{
    SlotHdr *hdr = reinterpret_cast<SlotHdr *>(slot ? slot + sl.o_hdr : nullptr);
    bool ok = slot != nullptr;
    uint32_t n = 0, n_lit = 0, blen = 0, n_extras = 0, onb = 1;
    if (ok) {
        ok = !(hdr->bad[LEN] | hdr->bad[OFF]);                         // the LIT stream is decoded later, on demand
        n = hdr->n_seq; n_lit = hdr->n_lit; blen = hdr->block_len; n_extras = hdr->n_extras; onb = hdr->off_nbytes;
        ok = ok && n <= sl.ms && onb >= 1 && onb <= 8;
    }
    if (!ok) n = 0;
    const uint32_t cq = ((n + 127) / 128) * 32;                        // sequences per warp, a multiple of 32
    const uint32_t k0 = min(n, r * cq), k1 = min(n, k0 + cq);
    const uint16_t *len16 = reinterpret_cast<const uint16_t *>(slot ? slot + sl.o_len : nullptr);
    const uint8_t *off_s = slot ? slot + sl.o_off : nullptr;
    const uint16_t *extras = ok ? reinterpret_cast<const uint16_t *>(cv.payload + ((uint64_t)hdr->rec_lo | (uint64_t)hdr->rec_hi << 32) +
                                                                     hdr->extras_off) : nullptr;
    // ---- pass 0: escapes per quarter
    uint32_t esc = 0;
    for (uint32_t k = k0 + lane; k < k1; k += 32) { const uint32_t v = len16[k]; esc += ((v & 0xFFu) == 255) + ((v >> 8) == 255); }
    esc = __reduce_add_sync(0xFFFFFFFFu, esc);
    if (lane == 0) sq[r][0] = esc;
    __syncthreads();
    uint32_t e0 = 0, e_all = 0;
    for (uint32_t i = 0; i < 4; i++) { const uint32_t x = sq[i][0]; if (i < r) e0 += x; e_all += x; }
    bool bad = e_all != n_extras;                                      // quad-uniform; bounds every extras index below
    // ---- pass 1: length sums per quarter (true values through the escapes)
    uint32_t s_ll = 0, s_all = 0;
    if (!bad) {
        uint32_t e = e0;
        for (uint32_t kb = k0; kb < k1; kb += 32) {
            const uint32_t k = kb + lane;
            uint32_t ll = 0, ml = 0;
            if (k < k1) { const uint32_t v = len16[k]; ll = v & 0xFFu; ml = (v >> 8) + 4; }
            if (n_extras) {
                const uint32_t e_ll = ll == 255, e_ml = ml == 259;
                uint32_t etot;
                uint32_t ei = e + warp_excl_scan(e_ll + e_ml, lane, etot);
                e += etot;
                if (e_ll) ll = extras[ei++];
                if (e_ml) ml = (uint32_t)extras[ei] + 4;
            }
            s_ll += ll; s_all += ll + ml;
        }
        s_ll = __reduce_add_sync(0xFFFFFFFFu, s_ll);
        s_all = __reduce_add_sync(0xFFFFFFFFu, s_all);
    }
    if (lane == 0) { sq[r][1] = s_ll; sq[r][2] = s_all; }
    __syncthreads();
    uint32_t lp = 0, pos = 0, t_ll = 0, t_all = 0;
    for (uint32_t i = 0; i < 4; i++) { const uint32_t x = sq[i][1], y = sq[i][2]; if (i < r) { lp += x; pos += y; } t_ll += x; t_all += y; }
    if (!bad) bad = t_ll > n_lit || t_all + (n_lit - t_ll) != blen;    // quad-uniform; every position below is < 16384
    // ---- pass 2: scan, token arrays, per-match checks
    if (!bad && ok) {
        uint16_t *start = reinterpret_cast<uint16_t *>(slot + sl.o_start);
        uint16_t *dst = reinterpret_cast<uint16_t *>(slot + sl.o_dst);
        uint16_t *litpos = reinterpret_cast<uint16_t *>(slot + sl.o_litpos);
        uint64_t *srcv = reinterpret_cast<uint64_t *>(slot + sl.o_src);
        const uint64_t B0 = blk << kBlockLog2;
        const uint64_t src_mask = ~0ull >> (64 - 8 * onb);
        uint32_t e = e0;
        // loads of round i+1 are issued before round i is processed
        uint32_t v_nx = 0, w0_nx = 0, w1_nx = 0, w2_nx = 0;
        auto fetch = [&](uint32_t k) {
            v_nx = w0_nx = w1_nx = w2_nx = 0;
            if (k < k1) {
                v_nx = len16[k];
                const uint32_t *wp = reinterpret_cast<const uint32_t *>(off_s + ((k * onb) & ~3u));   // stays inside the slot
                w0_nx = wp[0]; w1_nx = wp[1]; w2_nx = wp[2];
            }
        };
        fetch(k0 + lane);
        bool mbad = false;
        for (uint32_t kb = k0; kb < k1; kb += 32) {
            const uint32_t k = kb + lane;
            const bool act = k < k1;
            const uint32_t v = v_nx, w0 = w0_nx, w1 = w1_nx, w2 = w2_nx;
            fetch(k + 32);
            uint32_t ll = 0, ml = 0;
            if (act) { ll = v & 0xFFu; ml = (v >> 8) + 4; }
            if (n_extras) {
                const uint32_t e_ll = ll == 255, e_ml = ml == 259;
                uint32_t etot;
                uint32_t ei = e + warp_excl_scan(e_ll + e_ml, lane, etot);
                e += etot;
                if (e_ll) ll = extras[ei++];
                if (e_ml) ml = (uint32_t)extras[ei] + 4;
            }
            uint32_t ptot;
            const uint32_t pre = warp_excl_scan(ll | (ll + ml) << 16, lane, ptot);   // sums validated: no overflow
            const uint32_t my_lp = lp + (pre & 0xFFFFu), my_st = pos + (pre >> 16);
            lp += ptot & 0xFFFFu; pos += ptot >> 16;
            if (act) {
                const uint32_t sh = ((k * onb) & 3u) * 8;
                const uint32_t lo = __funnelshift_r(w0, w1, sh), hi = __funnelshift_r(w1, w2, sh);
                const uint64_t src = (((uint64_t)hi << 32) | lo) & src_mask;
                start[k] = (uint16_t)my_st;
                litpos[k] = (uint16_t)my_lp;
                dst[k] = (uint16_t)(my_st + ll);
                srcv[k] = src;
                if (src + ml > B0 + my_st + ll) mbad = true;           // strictly before, non-overlapping
            }
        }
        if (__any_sync(0xFFFFFFFFu, mbad)) bad = true;
        if (r == 3 && lane == 0) { start[n] = (uint16_t)t_all; litpos[n] = (uint16_t)t_ll; }
    }
    if (lane == 0) sq[r][3] = bad ? 1u : 0u;
    __syncthreads();
    if (slot && r == 0 && lane == 0) {
        const bool good = ok && !(sq[0][3] | sq[1][3] | sq[2][3] | sq[3][3]);
        if (ok && !good) raise(ctl, kStTokens, blk);
        hdr->parsed_ok = good ? 1u : 0u;
    }
    __syncthreads();                                                   // sq is reused by the next call
}

struct SeekArgs {
    uint64_t *pend;          // [nt][16384] per target byte: kDone | literal request | absolute position being chased
    uint32_t *mark;          // [n_blocks] claim word: the tag of the round that claimed the block
    unsigned long long *slot_of;   // [n_blocks] tag << 32 | slot, written by the claimer right after it won
    uint64_t *list;
    const uint64_t *ids;     // nt target ids (device); nullptr: the consecutive targets one_id, one_id + 1, ...
    uint64_t one_id;
    uint64_t range_lo;       // range mode: first byte of the range being decoded (see chase_byte)
    uint8_t *slots;
    uint8_t *out;
    uint64_t out_base;       // packed mode: target i lands at out + (out_base + i) * 16384
    uint32_t nt, absolute, max_slots;
    uint32_t tag0;           // round r marks the blocks it claims with tag0 + r
    uint32_t max_hops;
    uint32_t range_mode;     // 1: only bytes whose match source starts below range_lo are chased and written
};

constexpr unsigned long long kLitReq = 1ull << 62;   // pend = kLitReq | slot << 14 | index into the slot's LIT stream

__device__ inline uint64_t seek_target(const SeekArgs &a, uint32_t i) { return a.ids ? a.ids[i] : a.one_id + i; }

// Claim a slot of round `tag` for block blk (once: the claim word decides the winner). The slot entry
// carries the tag, so a reader can never pair a fresh claim with a stale slot index.
__device__ inline void claim_block(const SeekArgs &a, Control *ctl, uint32_t tag, uint32_t rp, uint64_t blk)
{
    if (a.mark[blk] == tag) return;
    if (atomicExch(a.mark + blk, tag) == tag) return;                  // somebody else claimed it
    const uint32_t s = atomicAdd(&ctl->round_n_list[rp], 1u);
    a.slot_of[blk] = (unsigned long long)tag << 32 | s;                // s >= max_slots: no slot in this round
    if (s < a.max_slots) a.list[s] = blk;
}

// Follow one byte through the parsed blocks that hold a slot in this round (slot entry of this round's
// tag with an index below n_ready, i.e. decoded and parsed before the last barrier) until it reaches a
// literal (-> literal request), leaves the resident set (-> stays a position; its block is claimed on the
// spot, for the next hop) or hits an inconsistency (-> kDone + status). Entries written during the
// current phase have an index >= n_ready, and a stale cached entry can only carry an older tag: both
// read as "not resident", which is always safe.
//
// Range mode (aceapex_decode_range): the targets are the consecutive blocks of a range whose other
// bytes the match kernel produces from the output buffer. A byte still at its OWN position (`own`) is at its first
// step: a literal, or a match whose source starts at or above range_lo, is left to the match kernel (kDone, nothing
// is written); a match whose source starts below the range is followed to its origin like any isolated byte.
__device__ inline unsigned long long chase_byte(const SlotLayout &sl, const SeekArgs &a, Control *ctl, uint32_t tag,
                                                uint32_t rp, uint32_t n_ready, unsigned long long p, unsigned long long own)
{
    bool first_step = a.range_mode && p == own;
    for (;;) {
        const uint64_t blk = p >> kBlockLog2;
        const uint32_t o = (uint32_t)(p & (kB - 1));
        const unsigned long long e = a.slot_of[blk];
        const uint32_t s = (uint32_t)e;
        if ((uint32_t)(e >> 32) != tag || s >= n_ready) { claim_block(a, ctl, tag, rp, blk); return p; }
        uint8_t *slot = a.slots + (size_t)s * sl.stride;
        SlotHdr *h = reinterpret_cast<SlotHdr *>(slot + sl.o_hdr);
        if (!h->parsed_ok) { raise(ctl, kStChase, blk); return kDone; }   // corrupt block: give up on this byte
        const uint32_t n = h->n_seq, blen = h->block_len;
        if (o >= blen) { raise(ctl, kStChase, blk); return kDone; }
        const uint16_t *start = reinterpret_cast<const uint16_t *>(slot + sl.o_start);
        uint32_t lo = 0, hi = n;                                       // largest q in [0, n] with start[q] <= o
        while (lo < hi) {
            const uint32_t mid = (lo + hi + 1) >> 1;
            if (start[mid] <= o) lo = mid; else hi = mid - 1;
        }
        const uint32_t q = lo, st = start[q];
        const uint32_t d = q < n ? reinterpret_cast<const uint16_t *>(slot + sl.o_dst)[q] : blen;
        if (o < d) {                                                   // a literal: the origin
            if (first_step) return kDone;
            const uint32_t li = (uint32_t)reinterpret_cast<const uint16_t *>(slot + sl.o_litpos)[q] + (o - st);
            if (li >= kB) { raise(ctl, kStChase, blk); return kDone; }
            h->need_lit = 1;
            return kLitReq | (unsigned long long)s << kBlockLog2 | li;
        }
        const unsigned long long src = reinterpret_cast<const uint64_t *>(slot + sl.o_src)[q];
        if (first_step && src >= a.range_lo) return kDone;
        first_step = false;
        const unsigned long long nxt = src + (o - d);                 // a match
        if (nxt >= p) { raise(ctl, kStChase, blk); return kDone; }
        p = nxt;
    }
}

// The fused kernel. CTAs of kEntropyWarps warps (the entropy phases need the per-warp tables), all
// co-resident. A ROUND keeps every block it touches resident in a slot:
//   chase hops:  collect the blocks of the bytes still chasing -> entropy-decode the LEN and OFF streams
//                of the NEW blocks (short streams) -> parse them -> follow every byte through all resident
//                blocks until it lands on a literal (a literal request: slot + index) or leaves them;
//   until nothing is chasing (or the slots are used up); then ONE literal phase:
//   entropy-decode the LIT stream of the slots that received a literal request, deliver the bytes.
// A seek therefore pays for the long LIT streams once, not once per hop, and ends on the device.
__global__ void __launch_bounds__(32 * kEntropyWarps, 2) k_seek_fused(Container cv, SlotLayout sl, SeekArgs a, Control *ctl)
{
    extern __shared__ __align__(1024) uint8_t smem_entropy[];
    __shared__ uint32_t s_rem;
    __shared__ uint32_t s_quad[kEntropyWarps / 4][4][4];
    const uint32_t lane = lane_id(), warp = threadIdx.x >> 5;
    WarpSmem ws;
    {
        const uint32_t a0 = (uint32_t)__cvta_generic_to_shared(smem_entropy);
        const uint32_t pad = (0u - a0) & (kT8Bytes - 1);
        uint8_t *base = smem_entropy + pad;
        ws.t8 = base + warp * kT8Bytes;
        ws.syml = reinterpret_cast<uint2 *>(base + kEntropyWarps * kT8Bytes + warp * kSymlBytes);
        ws.ring = base + kEntropyWarps * (kT8Bytes + kSymlBytes) + warp * kRingBytes;
        ws.a_t8 = (uint32_t)__cvta_generic_to_shared(ws.t8);
        ws.a_syml = (uint32_t)__cvta_generic_to_shared(ws.syml);
        ws.a_ring = (uint32_t)__cvta_generic_to_shared(ws.ring);
    }
    const uint32_t n_ctas = gridDim.x;
    const uint64_t n_thr = (uint64_t)n_ctas * blockDim.x, gtid = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    // Warp numbering CTA-minor: consecutive work items go to different SMs, so a seek that touches a few hundred
    // blocks runs one or two stream decodes per SM (each near its single-warp latency) instead of sixteen on a few SMs.
    const uint32_t n_warps = n_ctas * kEntropyWarps, gwarp = warp * n_ctas + blockIdx.x;
    const uint64_t n_bytes = (uint64_t)a.nt * kB;

    // init: every target byte chases its own position; the first round's claims are the targets themselves
    for (uint64_t g = gtid; g < n_bytes; g += n_thr) {
        const uint64_t id = seek_target(a, (uint32_t)(g >> kBlockLog2));
        const uint32_t o = (uint32_t)(g & (kB - 1));
        a.pend[g] = (id < cv.n_blocks && o < block_len_of(cv, id)) ? (id << kBlockLog2) + o : kDone;
    }
    for (uint64_t i = gtid; i < a.nt; i += n_thr) {
        const uint64_t id = seek_target(a, (uint32_t)i);
        if (id < cv.n_blocks) claim_block(a, ctl, a.tag0, 0, id);
    }
    grid_barrier();

    uint32_t hop = 0;
    for (uint32_t round = 0;; round++) {
        const uint32_t rp = round & 1u, tag = a.tag0 + round;
        uint32_t n_ready = 0;                                          // slots of this round decoded and parsed
        unsigned long long chasing = 0;
        // ---- round start (after the first): claim a slot for every distinct block a chasing byte sits in (later
        //      hops claim on the spot, at the end of their chase)
        if (round) {
            for (uint64_t g = gtid; g < n_bytes; g += n_thr) {
                const uint64_t p = a.pend[g];
                if (p < kLitReq) claim_block(a, ctl, tag, rp, p >> kBlockLog2);
            }
            grid_barrier();
        }
        for (;; hop++) {
            const uint32_t hp = hop & 1u;
            const uint32_t n_claimed = ld_acquire_u32(&ctl->round_n_list[rp]);
            const uint32_t n_now = n_claimed < a.max_slots ? n_claimed : a.max_slots;
            // ---- entropy: LEN and OFF of the new blocks, warp per (block, stream) unit
            const uint32_t n_new = n_now - n_ready;
            for (uint32_t u = gwarp; u < 2 * n_new; u += n_warps) {
                const uint32_t so = u / n_new, bi = n_ready + (u - so * n_new);
                if (so == 1 && lane == 0) reinterpret_cast<SlotHdr *>(a.slots + (size_t)bi * sl.stride + sl.o_hdr)->need_lit = 0;
                decode_unit(cv, sl, a.slots, a.list[bi], bi, so == 0 ? OFF : LEN, so == 1, ws, lane, ctl);
            }
            grid_barrier();
            if (gtid == 0) {                                           // the other parities' counters are idle now
                ctl->hop_pending[hp ^ 1u] = 0;
                if (n_ready == 0) ctl->round_n_list[rp ^ 1u] = 0;
            }
            // ---- parse the new blocks, four warps per block
            for (uint32_t b0 = n_ready + blockIdx.x * (kEntropyWarps / 4); b0 < n_now; b0 += n_ctas * (kEntropyWarps / 4)) {
                const uint32_t bi = b0 + (warp >> 2);
                uint8_t *slot = bi < n_now ? a.slots + (size_t)bi * sl.stride : nullptr;
                quad_parse_block(cv, sl, slot, slot ? a.list[bi] : 0, ctl, lane, warp & 3u, s_quad[warp >> 2]);
            }
            grid_barrier();
            n_ready = n_now;
            // ---- chase every byte through the resident blocks
            if (threadIdx.x == 0) s_rem = 0;
            __syncthreads();
            uint32_t remaining = 0;
            for (uint64_t g = gtid; g < n_bytes; g += n_thr) {
                const unsigned long long p = a.pend[g];
                if (p >= kLitReq) continue;
                const unsigned long long own = (seek_target(a, (uint32_t)(g >> kBlockLog2)) << kBlockLog2) + (g & (kB - 1));
                const unsigned long long q = chase_byte(sl, a, ctl, tag, rp, n_ready, p, own);
                if (q != p) a.pend[g] = q;
                remaining += q < kLitReq;
            }
            remaining = __reduce_add_sync(0xFFFFFFFFu, remaining);
            if (lane == 0 && remaining) atomicAdd(&s_rem, remaining);
            __syncthreads();
            if (threadIdx.x == 0 && s_rem) atomicAdd(&ctl->hop_pending[hp], (unsigned long long)s_rem);
            grid_barrier();
            chasing = ctl->hop_pending[hp];
            // out of slots: the blocks claimed beyond max_slots wait for the next round
            if (chasing == 0 || n_claimed >= a.max_slots || hop + 1 >= a.max_hops) { hop++; break; }
        }
        // ---- literal phase: LIT stream of every slot with a request, then deliver
        for (uint32_t bi = gwarp; bi < n_ready; bi += n_warps) {
            const SlotHdr *h = reinterpret_cast<const SlotHdr *>(a.slots + (size_t)bi * sl.stride + sl.o_hdr);
            if (h->need_lit && h->parsed_ok) decode_unit(cv, sl, a.slots, a.list[bi], bi, LIT, false, ws, lane, ctl);
        }
        grid_barrier();
        for (uint64_t g = gtid; g < n_bytes; g += n_thr) {
            const unsigned long long p = a.pend[g];
            if (p == kDone || p < kLitReq) continue;
            const uint32_t s = (uint32_t)((p ^ kLitReq) >> kBlockLog2), li = (uint32_t)(p & (kB - 1));
            const uint8_t *slot = a.slots + (size_t)s * sl.stride;
            const SlotHdr *h = reinterpret_cast<const SlotHdr *>(slot + sl.o_hdr);
            if (!h->bad[LIT] && li < h->n_lit) {
                const uint32_t i = (uint32_t)(g >> kBlockLog2);
                a.out[((a.absolute ? seek_target(a, i) : a.out_base + i) << kBlockLog2) + (g & (kB - 1))] = slot[sl.o_lit + li];
            } else {
                raise(ctl, kStChase, a.list[s]);
            }
            a.pend[g] = kDone;
        }
        if (chasing == 0) break;
        if (hop >= a.max_hops) {                                       // deeper than this build follows a chain
            if (gtid == 0) raise(ctl, kStChase, 0);
            break;
        }
        grid_barrier();                                     // the slots are recycled by the next round
    }
    // leave the counters of both parities at zero for the next call
    grid_barrier();
    if (gtid == 0) {
        ctl->round_n_list[0] = ctl->round_n_list[1] = 0;
        ctl->hop_pending[0] = ctl->hop_pending[1] = 0;
    }
}

}  // namespace aceapex
