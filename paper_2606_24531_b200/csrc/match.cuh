// Match layer: token parse (FORMAT.md section 4), literal placement and absolute-offset copies
// (PAPER.md:19, :27), with cross-block ordering by ticket + watermark ("any block decodes once
// the blocks holding its source bytes are present").
#pragma once
#include "entropy.cuh"

namespace aceapex {

constexpr uint32_t kMatchThreads = 256;
constexpr uint32_t kMatchWarps = kMatchThreads / 32;

// Token arrays of one block (shared memory in decode_all, the slot in the isolated path).
struct Tokens {
    uint16_t *start;   // [n_seq+1] in-block output offset where sequence k's literal run starts;
                       //           entry n_seq = start of the trailing literals
    uint16_t *dst;     // [n_seq]   in-block output offset of match k
    uint16_t *litpos;  // [n_seq+1] index into LIT of sequence k's first literal
    uint64_t *src;     // [n_seq]   absolute source position of match k
    uint32_t *bm;      // optional [512]: bit o set iff some sequence (or the trailing run) starts at offset o
};

// Exclusive prefix sum of one value per thread over the CTA (kMatchThreads threads).
__device__ inline uint32_t block_excl_scan(uint32_t v, uint32_t *warp_sums /* [kMatchWarps+1] smem */,
                                           uint32_t &total)
{
    const uint32_t lane = lane_id(), warp = threadIdx.x >> 5;
    uint32_t wtotal;
    const uint32_t in_warp = warp_excl_scan(v, lane, wtotal);
    __syncthreads();                       // warp_sums may still be read from a previous scan
    if (lane == 0) warp_sums[warp] = wtotal;
    __syncthreads();
    uint32_t base = 0, tot = 0;
#pragma unroll
    for (uint32_t w = 0; w < kMatchWarps; w++) {
        const uint32_t t = warp_sums[w];
        if (w < warp) base += t;
        tot += t;
    }
    total = tot;
    return base + in_warp;
}

// Parse the decoded LEN / OFF streams of a block into token arrays (FORMAT.md section 4).
// All kMatchThreads threads of the CTA call this. Returns true (CTA-uniform) iff every validity
// rule holds: escapes consumed == n_extras, sum lit_len <= n_lit, sums == block_len, and for every
// match src + match_len <= dst (absolute) — after which every copy below is in bounds.
__device__ inline bool parse_tokens(const Record &r, uint64_t blk, const uint8_t *len_s, const uint8_t *off_s,
                                    const Tokens &t, uint32_t *warp_sums, uint64_t *max_src_blk_below)
{
    const uint32_t n = r.n_seq;
    const uint32_t per = (n + kMatchThreads - 1) / kMatchThreads;
    const uint32_t k0 = min(n, threadIdx.x * per), k1 = min(n, k0 + per);
    const uint16_t *extras = reinterpret_cast<const uint16_t *>(r.rec + r.extras_off);
    const uint64_t B0 = blk << kBlockLog2;

    uint32_t esc = 0;
    for (uint32_t k = k0; k < k1; k++) esc += (len_s[2 * k] == 255) + (len_s[2 * k + 1] == 255);
    uint32_t esc_total;
    const uint32_t esc_base = block_excl_scan(esc, warp_sums, esc_total);
    if (esc_total != r.n_extras) return false;               // CTA-uniform

    uint32_t sum_ll = 0, sum_all = 0;
    {
        uint32_t e = esc_base;
        for (uint32_t k = k0; k < k1; k++) {
            uint32_t ll = len_s[2 * k], ml = len_s[2 * k + 1];
            if (ll == 255) ll = extras[e++];
            if (ml == 255) ml = extras[e++];
            sum_ll += ll;
            sum_all += ll + ml + 4;
        }
    }
    uint32_t ll_total, all_total;
    const uint32_t ll_base = block_excl_scan(sum_ll, warp_sums, ll_total);
    const uint32_t all_base = block_excl_scan(sum_all, warp_sums, all_total);
    if (ll_total > r.n_lit) return false;
    if (all_total + (r.n_lit - ll_total) != r.block_len) return false;

    bool bad = false;
    uint64_t below = 0;                                      // 1 + highest earlier block read
    {
        uint32_t e = esc_base, lp = ll_base, pos = all_base;
        for (uint32_t k = k0; k < k1; k++) {
            uint32_t ll = len_s[2 * k], ml = len_s[2 * k + 1];
            if (ll == 255) ll = extras[e++];
            if (ml == 255) ml = extras[e++];
            ml += 4;
            uint64_t src = 0;
            for (uint32_t j = 0; j < r.off_nbytes; j++) src |= (uint64_t)off_s[k * r.off_nbytes + j] << (8 * j);
            t.start[k] = (uint16_t)pos;
            t.litpos[k] = (uint16_t)lp;
            if (t.bm && pos < kB) atomicOr(&t.bm[pos >> 5], 1u << (pos & 31));
            pos += ll; lp += ll;
            t.dst[k] = (uint16_t)pos;
            t.src[k] = src;
            if (src + ml > B0 + pos) bad = true;             // strictly before, non-overlapping
            if (src < B0) {
                const uint64_t last = (src + ml < B0 ? src + ml : B0) - 1;
                const uint64_t need = (last >> kBlockLog2) + 1;
                if (need > below) below = need;
            }
            pos += ml;
        }
    }
    if (threadIdx.x == kMatchThreads - 1) {
        t.start[n] = (uint16_t)all_total;
        t.litpos[n] = (uint16_t)ll_total;
        if (t.bm && all_total < kB) atomicOr(&t.bm[all_total >> 5], 1u << (all_total & 31));
    }
    if (max_src_blk_below) {
        // CTA-wide max via shared atomics; caller zeroed *max_src_blk_below before the call
        if (below) atomicMax(reinterpret_cast<unsigned long long *>(max_src_blk_below), (unsigned long long)below);
    }
    return !__syncthreads_or(bad);
}

// ---- cross-block ordering ---------------------------------------------------------------------

__device__ inline uint32_t ld_acquire_u32(const uint32_t *p)
{
    uint32_t v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ inline unsigned long long ld_acquire_u64(const unsigned long long *p)
{
    unsigned long long v;
    asm volatile("ld.acquire.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}
__device__ inline void st_release_u32(uint32_t *p, uint32_t v)
{
    asm volatile("st.release.gpu.global.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}

// Advance the watermark over every leading block whose done flag carries this call's epoch.
// Called by all 32 lanes of one warp: 32 flags are examined per round trip. Returns the new
// watermark (warp-uniform). The flags were read with acquire semantics and the fence orders them
// before the atomicMax, so whoever later acquires the watermark also sees those blocks' bytes.
__device__ inline unsigned long long advance_watermark(Control *ctl, const uint32_t *done, uint64_t n_blocks,
                                                       uint32_t epoch)
{
    const uint32_t lane = lane_id();
    unsigned long long w0 = 0;
    if (lane == 0) w0 = ld_acquire_u64(&ctl->watermark);
    w0 = __shfl_sync(0xFFFFFFFFu, w0, 0);
    unsigned long long w = w0;
    for (;;) {
        const unsigned long long idx = w + lane;
        const bool f = idx < n_blocks && ld_acquire_u32(done + idx) == epoch;
        const uint32_t m = __ballot_sync(0xFFFFFFFFu, f);
        const uint32_t c = m == 0xFFFFFFFFu ? 32u : (uint32_t)__ffs(~m) - 1u;
        w += c;
        if (c < 32) break;
    }
    if (w > w0 && lane == 0) {
        __threadfence();
        atomicMax(&ctl->watermark, w);
    }
    return w;
}

// Source byte of a match at absolute position p: inside the block from the tile, else from the
// output buffer (an earlier, completed block).
__device__ inline uint32_t src_byte(const uint8_t *tile, const uint8_t *out, uint64_t B0, uint64_t p)
{
    return p >= B0 ? tile[p - B0] : out[p];
}

// decode_all, match layer. One CTA per block; block ids are handed out in increasing order by a
// ticket, so a CTA only ever waits for blocks whose CTAs are already running or finished.
//   slots: decoded streams of blocks first .. first+count-1 (slot i = block first+i).
//
// Pass 0 is output-centric: every thread produces groups of 4 consecutive output bytes. The
// sequence that owns output offset o is rank[o>>5] + popc(bitmap word below o) - 1, where the
// bitmap marks the start offset of every sequence: no search. Literal bytes come from the LIT
// stream, bytes of tag-0 matches (source entirely in earlier blocks) from the output buffer.
// Matches with tag >= 1 (source inside this block) follow level by level (FORMAT.md section 4).
__global__ void __launch_bounds__(kMatchThreads) k_match(Container cv, SlotLayout sl, const uint8_t *slots,
                                                          uint64_t first, uint32_t count, uint8_t *out,
                                                          uint32_t out_aligned16, Control *ctl, uint32_t *done,
                                                          uint32_t epoch)
{
    extern __shared__ __align__(16) uint8_t smem[];
    __shared__ uint32_t warp_sums[kMatchWarps + 1];
    __shared__ uint32_t s_ticket;
    __shared__ unsigned long long s_below;
    __shared__ uint32_t s_maxtag;

    uint8_t *tile = smem;                                    // 16384
    uint32_t *bm = reinterpret_cast<uint32_t *>(smem + kB);  // 512 words
    uint16_t *rank = reinterpret_cast<uint16_t *>(smem + kB + 2048);   // 512
    Tokens t;
    t.src = reinterpret_cast<uint64_t *>(smem + kB + 3072);
    t.start = reinterpret_cast<uint16_t *>(smem + kB + 3072 + 8 * sl.ms);
    t.dst = t.start + (sl.ms + 16);
    t.litpos = t.dst + sl.ms;
    t.bm = bm;
    uint8_t *tags = reinterpret_cast<uint8_t *>(t.litpos + (sl.ms + 16));   // [ms]

    if (threadIdx.x == 0) {
        s_ticket = atomicAdd(&ctl->ticket, 1u);
        s_below = 0;
        s_maxtag = 0;
    }
    for (uint32_t i = threadIdx.x; i < 512; i += kMatchThreads) bm[i] = 0;
    __syncthreads();
    const uint32_t bi = s_ticket;
    if (bi < count) {
        const uint64_t blk = first + bi;
        const uint64_t B0 = blk << kBlockLog2;
        const uint8_t *slot = slots + (size_t)bi * sl.stride;
        const SlotHdr *hdr = reinterpret_cast<const SlotHdr *>(slot + sl.o_hdr);
        const Record r = open_record(cv, blk);
        bool ok = r.ok && !(hdr->bad[0] | hdr->bad[1] | hdr->bad[2]) && r.n_seq <= sl.ms;
        if (ok) {
            ok = parse_tokens(r, blk, slot + sl.o_len, slot + sl.o_off, t, warp_sums, (uint64_t *)&s_below);
            if (!ok && threadIdx.x == 0) raise(ctl, kStTokens, blk);
        }
        if (ok) {
            const uint32_t n = r.n_seq, blen = r.block_len;
            const uint8_t *lit = slot + sl.o_lit;
            const uint8_t *tagsec = r.rec + r.tags_off;
            uint32_t mt = 0;
            for (uint32_t k = threadIdx.x; k < n; k += kMatchThreads) {
                const uint32_t tg = (tagsec[k >> 1] >> ((k & 1) * 4)) & 15u;
                tags[k] = (uint8_t)tg;
                mt = max(mt, tg);
            }
            if (mt) atomicMax(&s_maxtag, mt);
            // rank[w] = number of sequence starts in bitmap words before w
            {
                uint32_t p0 = 0, p1 = 0, p2 = 0, p3 = 0;
                if (threadIdx.x < 128) {
                    const uint4 w = reinterpret_cast<const uint4 *>(bm)[threadIdx.x];
                    p0 = __popc(w.x); p1 = __popc(w.y); p2 = __popc(w.z); p3 = __popc(w.w);
                }
                uint32_t tot;
                const uint32_t r0 = block_excl_scan(p0 + p1 + p2 + p3, warp_sums, tot);
                if (threadIdx.x < 128)
                    reinterpret_cast<uint2 *>(rank)[threadIdx.x] =
                        make_uint2(r0 | (r0 + p0) << 16, (r0 + p0 + p1) | (r0 + p0 + p1 + p2) << 16);
            }
            // wait until every earlier block this block copies from is complete
            const uint32_t warp = threadIdx.x >> 5;
            const uint64_t below = s_below;                  // 1 + highest earlier block read
            if (below && warp == 0) {
                while (advance_watermark(ctl, done, cv.n_blocks, epoch) < below) __nanosleep(64);
                __threadfence();
            }
            __syncthreads();
            // pass 0: literals and tag-0 matches, 4 output bytes per thread per step
            for (uint32_t o = 4 * threadIdx.x; o < blen; o += 4 * kMatchThreads) {
                const uint32_t w = bm[o >> 5], sh = o & 31u;
                const uint32_t q = (uint32_t)rank[o >> 5] + __popc(w & ((2u << sh) - 1u)) - 1u;
                const uint32_t st = t.start[q], d = q < n ? t.dst[q] : blen;
                uint32_t v = 0;
                const bool one_seq = ((w >> sh) & 0xEu) == 0 && o + 4 <= blen;
                if (one_seq && o + 4 <= d) {                 // four literal bytes of sequence q
                    const uint8_t *p = lit + t.litpos[q] + (o - st);
                    v = p[0] | p[1] << 8 | p[2] << 16 | p[3] << 24;
                } else if (one_seq && o >= d) {              // four bytes of match q
                    if (tags[q] == 0) {
                        const uint8_t *p = out + t.src[q] + (o - d);
                        v = p[0] | p[1] << 8 | p[2] << 16 | p[3] << 24;
                    }
                } else {                                     // a boundary inside the group
                    uint32_t qq = q, s0 = st, dd = d;
                    for (uint32_t j = 0; j < 4 && o + j < blen; j++) {
                        const uint32_t oj = o + j;
                        if (j && ((w >> (sh + j)) & 1u)) { qq++; s0 = oj; dd = qq < n ? t.dst[qq] : blen; }
                        uint32_t b = 0;
                        if (oj < dd) b = lit[t.litpos[qq] + (oj - s0)];
                        else if (tags[qq] == 0) b = out[t.src[qq] + (oj - dd)];
                        v |= b << (8 * j);
                    }
                }
                *reinterpret_cast<uint32_t *>(tile + o) = v;
            }
            __syncthreads();
            // matches whose source lies (partly) inside this block, level by level
            const uint32_t maxtag = s_maxtag;
            for (uint32_t level = 1; level <= maxtag; level++) {
                for (uint32_t k = threadIdx.x; k < n; k += kMatchThreads) {
                    if (tags[k] != level) continue;
                    const uint32_t d = t.dst[k], ml = t.start[k + 1] - d;
                    const uint64_t src = t.src[k];
                    for (uint32_t j = 0; j < ml; j++) tile[d + j] = (uint8_t)src_byte(tile, out, B0, src + j);
                }
                __syncthreads();
            }
            // tile -> output
            uint8_t *dstp = out + B0;
            if (out_aligned16) {
                const uint32_t nvec = blen >> 4;
                const uint4 *tv = reinterpret_cast<const uint4 *>(tile);
                uint4 *ov = reinterpret_cast<uint4 *>(dstp);
                for (uint32_t i = threadIdx.x; i < nvec; i += kMatchThreads) ov[i] = tv[i];
                for (uint32_t i = (nvec << 4) + threadIdx.x; i < blen; i += kMatchThreads) dstp[i] = tile[i];
            } else {
                for (uint32_t i = threadIdx.x; i < blen; i += kMatchThreads) dstp[i] = tile[i];
            }
        } else if (threadIdx.x == 0 && !r.ok) {
            raise(ctl, kStRecord, blk);
        }
        // publish (also for a bad block: later blocks must not wait forever)
        __threadfence();
        __syncthreads();
        if (threadIdx.x < 32) {
            if (threadIdx.x == 0) st_release_u32(done + blk, epoch);
            __syncwarp();
            advance_watermark(ctl, done, cv.n_blocks, epoch);
        }
    }
    // last CTA out re-arms the ticket for the next launch
    if (threadIdx.x == 0) {
        __threadfence();
        if (atomicAdd(&ctl->ticket_exit, 1u) == gridDim.x - 1) {
            ctl->ticket = 0;
            ctl->ticket_exit = 0;
            __threadfence();
        }
    }
}

// Isolated path: parse the tokens of every listed block into its slot (global memory).
__global__ void __launch_bounds__(kMatchThreads) k_parse(Container cv, SlotLayout sl, uint8_t *slots,
                                                          const uint64_t *list, const uint32_t *n_list,
                                                          uint32_t max_slots, Control *ctl)
{
    __shared__ uint32_t warp_sums[kMatchWarps + 1];
    uint32_t nb = *n_list;
    if (nb > max_slots) nb = max_slots;
    for (uint32_t bi = blockIdx.x; bi < nb; bi += gridDim.x) {
        const uint64_t blk = list[bi];
        uint8_t *slot = slots + (size_t)bi * sl.stride;
        SlotHdr *hdr = reinterpret_cast<SlotHdr *>(slot + sl.o_hdr);
        const Record r = open_record(cv, blk);
        bool ok = r.ok && !(hdr->bad[0] | hdr->bad[1] | hdr->bad[2]) && r.n_seq <= sl.ms;
        Tokens t;
        t.start = reinterpret_cast<uint16_t *>(slot + sl.o_start);
        t.dst = reinterpret_cast<uint16_t *>(slot + sl.o_dst);
        t.litpos = reinterpret_cast<uint16_t *>(slot + sl.o_litpos);
        t.src = reinterpret_cast<uint64_t *>(slot + sl.o_src);
        t.bm = nullptr;
        if (ok) {
            ok = parse_tokens(r, blk, slot + sl.o_len, slot + sl.o_off, t, warp_sums, nullptr);
            if (!ok && threadIdx.x == 0) raise(ctl, kStTokens, blk);
        }
        if (threadIdx.x == 0) {
            hdr->n_seq = r.n_seq;
            hdr->n_lit = r.n_lit;
            hdr->block_len = r.block_len;
            hdr->parsed_ok = ok ? 1u : 0u;
        }
        __syncthreads();
    }
}

}  // namespace aceapex
