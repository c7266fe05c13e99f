// Match layer: token parse (FORMAT.md section 4), literal placement and absolute-offset copies
// (PAPER.md:19, :27), with cross-block ordering by ticket + watermark ("any block decodes once
// the blocks holding its source bytes are present").
#pragma once
#include "entropy.cuh"

namespace aceapex {

constexpr uint32_t kMatchThreads = 256;
constexpr uint32_t kMatchWarps = kMatchThreads / 32;

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

// Cross-block ordering. A finished block publishes its done flag (epoch of this call) with release
// semantics; the flag store follows the CTA barrier that ends the block's writes, and a release is
// cumulative over what the barrier ordered before it, so one thread publishes for the whole CTA.
// The watermark (number of leading complete blocks) is kept moving by a helper CTA (ticket 0 of the
// match kernel), which scans the done flags with acquire loads and publishes the new value with a
// fence + atomicMax, so that whoever later acquires the watermark also sees those blocks' bytes.
// A block reads the watermark once, early; if that value does not cover its highest source block yet
// (no window promise, or the helper lags), its first warp scans the flags itself with the function
// below - correct for any valid stream, with or without the helper. Block ids are handed out in
// increasing order, so every block a CTA waits for belongs to a CTA that is running or finished: no
// deadlock.
//   blocking = false stops at the first incomplete block instead of spinning (the helper's mode).
__device__ inline unsigned long long wait_for_blocks(Control *ctl, const uint32_t *done, uint32_t epoch,
                                                     unsigned long long w, unsigned long long below, bool blocking)
{
    const uint32_t lane = lane_id();
    const unsigned long long w0 = w;
    while (w < below) {
        const unsigned long long idx = w + lane;
        const bool f = idx >= below || ld_acquire_u32(done + idx) == epoch;
        const uint32_t m = __ballot_sync(0xFFFFFFFFu, f);
        if (m == 0xFFFFFFFFu) {
            w = w + 32 < below ? w + 32 : below;
        } else {
            w += (uint32_t)__ffs(~m) - 1u;
            if (!blocking) break;
            __nanosleep(200);
        }
    }
    if (w > w0 && lane == 0) {
        __threadfence();
        atomicMax(&ctl->watermark, w);
    }
    return w;
}

// ---- decode_all match kernel --------------------------------------------------------------------
//
// Output-centric and branch-free. After the parse every output byte belongs to exactly one *run*:
// the literal run of sequence q (run index 2q+1), the match of sequence q (2q+2) or the trailing
// literals (2n+1). Two bitmaps over the 16,384 output offsets mark where sequences start (S) and
// where matches start (D); the run that owns offset o is
//     r(o) = #S bits <= o  +  #D bits <= o          (a rank word + two popcounts, no search)
// and its source byte sits at address delta[r] + o, where delta[r] is
//     literal run: &LIT[litpos_q] - start_q          (decoded LIT stream in the slot)
//     match:       &out[src_q]   - dst_q             (absolute offset into the output buffer)
// so literals and copies are the same instruction sequence: one 8-byte table load and one byte load
// per output byte, four bytes per thread per step, one 32-bit store straight to the output buffer
// (no staging tile: in-block sources are read back from the output buffer as well, which gives
// cross-block and in-block copies one address space).
//
// Matches with tag >= 1 (source range reaches into this block, FORMAT.md section 4) are produced
// by pass 0 with whatever the buffer held and then rewritten level by level from a list sorted by tag.

#ifdef ACEAPEX_TRACE
__device__ unsigned long long g_trace[16];
#define TRACE_MARK(i) do { if (threadIdx.x == 0) { const long long t_ = clock64(); atomicAdd(&g_trace[i], (unsigned long long)(t_ - t_prev)); t_prev = t_; } } while (0)
#define TRACE_DECL long long t_prev = clock64()
#else
#define TRACE_MARK(i) do { } while (0)
#define TRACE_DECL do { } while (0)
#endif

constexpr uint32_t kMatchFixedSmem = 4096 + 1024 + 16;   // bm2 + rk + delta[0] pad (delta[1] is 16-byte aligned)

__host__ __device__ inline uint32_t match_smem_bytes(uint32_t ms, uint32_t W)
{
    // delta (16 ms + 16), dm (4 ms), tlist (2 ms), staged LEN / slist (2 ms), staged OFF (W ms + 16: the
    // word-wise offset read may touch 11 bytes past the last offset), staged tags (ms / 2)
    return kMatchFixedSmem + 16 * ms + 16 + 4 * ms + 2 * ms + 2 * ms + (W * ms + 16) + ((ms / 2 + 15u) & ~15u);
}

__device__ inline uint32_t ldg_u8(unsigned long long a)
{
    uint32_t v;
    asm volatile("ld.global.u8 %0, [%1];" : "=r"(v) : "l"(a) : "memory");
    return v;
}

// Exclusive prefix sums of two values per thread over the CTA.
__device__ inline void block_excl_scan2(uint32_t a, uint32_t b, uint32_t (*ws)[2] /* [kMatchWarps] smem */,
                                        uint32_t &ea, uint32_t &eb, uint32_t &ta, uint32_t &tb)
{
    const uint32_t lane = lane_id(), warp = threadIdx.x >> 5;
    uint32_t wa, wb;
    const uint32_t ia = warp_excl_scan(a, lane, wa), ib = warp_excl_scan(b, lane, wb);
    __syncthreads();
    if (lane == 0) { ws[warp][0] = wa; ws[warp][1] = wb; }
    __syncthreads();
    uint32_t ba = 0, bb = 0, sa = 0, sb = 0;
#pragma unroll
    for (uint32_t w = 0; w < kMatchWarps; w++) {
        const uint32_t xa = ws[w][0], xb = ws[w][1];
        if (w < warp) { ba += xa; bb += xb; }
        sa += xa; sb += xb;
    }
    ea = ba + ia; eb = bb + ib; ta = sa; tb = sb;
}

// The four source addresses of output bytes o .. o+3 (o a multiple of 4).
struct Addr4 { unsigned long long a0, a1, a2, a3; };
__device__ inline Addr4 run_addresses(const uint2 *bm2, const uint16_t *rk, const unsigned long long *delta, uint32_t o)
{
    const uint2 w = bm2[o >> 5];
    const uint32_t sh = o & 31u, m = (2u << sh) - 1u;
    const uint32_t r0 = (uint32_t)rk[o >> 5] + __popc(w.x & m) + __popc(w.y & m);
    const uint32_t t = w.x >> sh, u = w.y >> sh;
    const uint32_t r1 = r0 + ((t >> 1) & 1u) + ((u >> 1) & 1u);
    const uint32_t r2 = r1 + ((t >> 2) & 1u) + ((u >> 2) & 1u);
    const uint32_t r3 = r2 + ((t >> 3) & 1u) + ((u >> 3) & 1u);
    // Most groups lie in one run or straddle one boundary: the first and the last entry are always
    // loaded, the middle ones only when they differ from both (the shared-memory pipe is the busy one).
    const unsigned long long d0 = delta[r0], d3 = delta[r3];
    unsigned long long d1 = r1 == r0 ? d0 : d3, d2 = r2 == r0 ? d0 : d3;
    if (r1 != r0 && r1 != r3) d1 = delta[r1];
    if (r2 != r0 && r2 != r3) d2 = delta[r2];
    Addr4 a;
    a.a0 = d0 + o;
    a.a1 = d1 + o + 1;
    a.a2 = d2 + o + 2;
    a.a3 = d3 + o + 3;
    return a;
}

__device__ inline uint32_t ldg_u32(unsigned long long a)
{
    uint32_t v;
    asm volatile("ld.global.u32 %0, [%1];" : "=r"(v) : "l"(a) : "memory");
    return v;
}

// Word-granular plan of output bytes o .. o+3: the run of byte 0 (source address aA for byte 0), the
// position k of the first run boundary inside the group (4 = none), the run of byte 3 (source address
// aB for byte k) and whether there is a second boundary (then the group takes the per-byte path).
// With at most one boundary the four bytes are k bytes at aA.. and 4-k bytes at aB..: two (unaligned)
// 32-bit windows, each fetched as one or two ALIGNED words instead of four byte loads that touch the
// same cache lines four times.
#ifndef ACEAPEX_WORD_UNROLL
#define ACEAPEX_WORD_UNROLL 4
#endif
constexpr uint32_t kWordUnroll = ACEAPEX_WORD_UNROLL;   // steps whose loads are in flight together
struct GroupPlan { unsigned long long aA, aB; uint32_t k, multi; };
__device__ inline GroupPlan plan_group(const uint2 *bm2, const uint16_t *rk, const unsigned long long *delta, uint32_t o)
{
    const uint2 w = bm2[o >> 5];
    const uint32_t sh = o & 31u, m = (2u << sh) - 1u;
    const uint32_t r0 = (uint32_t)rk[o >> 5] + __popc(w.x & m) + __popc(w.y & m);
    const uint32_t t = (w.x >> sh) & 0xEu, u = (w.y >> sh) & 0xEu, x = t | u;
    const uint32_t r3 = r0 + __popc(t) + __popc(u);                    // run of byte 3 (of byte k when there is one boundary)
    GroupPlan g;
    g.k = x ? (uint32_t)__ffs(x) - 1u : 4u;
    g.multi = (x & (x - 1u)) != 0;
    g.aA = delta[r0] + o;
    g.aB = delta[r3] + o + (g.k & 3u);
    return g;
}

__device__ inline void store4(unsigned long long a, uint32_t v, uint32_t aligned4)
{
    if (aligned4) {
        asm volatile("st.global.u32 [%0], %1;" ::"l"(a), "r"(v) : "memory");
    } else {
        asm volatile("st.global.u8 [%0], %1;" ::"l"(a), "r"(v) : "memory");
        asm volatile("st.global.u8 [%0], %1;" ::"l"(a + 1), "r"(v >> 8) : "memory");
        asm volatile("st.global.u8 [%0], %1;" ::"l"(a + 2), "r"(v >> 16) : "memory");
        asm volatile("st.global.u8 [%0], %1;" ::"l"(a + 3), "r"(v >> 24) : "memory");
    }
}

__global__ void __launch_bounds__(kMatchThreads) k_match(Container cv, SlotLayout sl, const uint8_t *slots,
                                                          uint64_t first, uint32_t count, uint8_t *out,
                                                          uint32_t out_aligned4, Control *ctl, uint32_t *done,
                                                          uint32_t epoch)
{
    extern __shared__ __align__(16) uint8_t smem[];
    __shared__ uint32_t ws3[kMatchWarps][3];
    __shared__ uint32_t ws2[kMatchWarps][2];
    __shared__ uint32_t s_ticket, s_ntag, s_bad, s_below;
    __shared__ unsigned long long s_wm;
    __shared__ uint32_t s_cnt[16], s_cur[16];

    const uint32_t ms = sl.ms;
    uint2 *bm2 = reinterpret_cast<uint2 *>(smem);                                   // [512] {S word, D word}
    uint16_t *rk = reinterpret_cast<uint16_t *>(smem + 4096);                       // [512]
    unsigned long long *delta = reinterpret_cast<unsigned long long *>(smem + 4096 + 1024 + 8);   // [2*ms+2]
    uint32_t *dm = reinterpret_cast<uint32_t *>(smem + kMatchFixedSmem + 16 * ms + 16);          // [ms] dst | len << 16
    uint16_t *tlist = reinterpret_cast<uint16_t *>(dm + ms);                        // [ms] k | tag << 12, unsorted
    uint16_t *s_len16 = tlist + ms;                                                 // [ms] staged LEN stream (u8 pairs)
    uint16_t *slist = s_len16;                                                      // [ms] tag list sorted by tag (after the parse)
    uint8_t *s_off = reinterpret_cast<uint8_t *>(s_len16 + ms);                     // [W*ms] staged OFF stream
    uint8_t *s_tags = s_off + cv.W * ms + 16;                                            // [ms/2] staged tag nibbles

    const uint32_t tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5;
    const uint32_t lt = (1u << lane) - 1u;
  // Persistent CTAs: each takes block after block from the ticket counter until none is left.
  for (;;) {
    __syncthreads();                                                   // the previous block's shared state is dead
    if (tid == 0) {
        s_ticket = atomicAdd(&ctl->ticket, 1u);
        s_below = 0;
        s_ntag = 0;
        s_bad = 0;
    }
    if (tid < 16) s_cnt[tid] = 0;
    for (uint32_t i = tid; i < 256; i += kMatchThreads) reinterpret_cast<uint4 *>(bm2)[i] = make_uint4(0, 0, 0, 0);
    __syncthreads();
    if (s_ticket > count) break;                                       // tickets 1 .. count are blocks
    TRACE_DECL;
    if (s_ticket == 0) {
        // Ticket 0 (a CTA that is certainly running) does not decode a block: its first warp keeps the
        // watermark moving for everybody, 32 done flags per round trip, until this launch's blocks are done.
        const unsigned long long end = first + count;
        if (tid == 0) s_wm = ld_acquire_u64(&ctl->watermark);
        __syncthreads();
        unsigned long long w = s_wm;
        while (w < end) {
            const unsigned long long idx = w + tid;
            const bool f = idx >= end || ld_acquire_u32(done + idx) == epoch;
            const uint32_t m = __ballot_sync(0xFFFFFFFFu, f);
            if (lane == 0) ws2[warp][0] = m == 0xFFFFFFFFu ? 32u : (uint32_t)__ffs(~m) - 1u;
            __syncthreads();
            uint32_t lead = 0;
#pragma unroll
            for (uint32_t i = 0; i < kMatchWarps; i++) {
                const uint32_t c = ws2[i][0];
                if (lead == 32 * i) lead += c;                         // only while every earlier warp was complete
            }
            __syncthreads();
            if (lead) {
                w = w + lead < end ? w + lead : end;
                if (tid == 0) { __threadfence(); atomicMax(&ctl->watermark, w); }
            } else {
                __nanosleep(300);
            }
        }
    }
    const uint32_t bi = s_ticket - 1;                                  // ticket 0 -> 0xFFFFFFFF: no block
    if (bi < count) {
        const uint64_t blk = first + bi;
        const uint64_t B0 = blk << kBlockLog2;
        const uint8_t *slot = slots + (size_t)bi * sl.stride;
        // the record header fields as the entropy kernel's LIT unit left them in the slot header
        struct { const uint8_t *rec; uint32_t n_seq, n_lit, block_len, n_extras, off_nbytes, extras_off, tags_off; bool ok; } r;
        {
            const uint4 *hp = reinterpret_cast<const uint4 *>(slot + sl.o_hdr);
            const uint4 h0 = hp[0], h1 = hp[1], h2 = hp[2], h3 = hp[3];
            r.ok = !(h0.x | h0.y | h0.z);                              // bad[LIT] covers an invalid record header
            r.n_seq = h0.w; r.n_lit = h1.x; r.block_len = h1.y;
            r.n_extras = h1.w; r.off_nbytes = h2.x; r.extras_off = h2.y; r.tags_off = h2.z;
            r.rec = cv.payload + ((uint64_t)h2.w | (uint64_t)h3.x << 32);
        }
        bool ok = r.ok && r.n_seq <= ms;
        const uint32_t n = ok ? r.n_seq : 0, blen = ok ? r.block_len : 0;
        TRACE_MARK(0);
        if (ok) {
            // ---- parse (FORMAT.md section 4). Warp w owns the sequences [w*cw, (w+1)*cw), lane-strided:
            // in round i lane l holds sequence w*cw + 32*i + l, so loads coalesce and the prefix sums are
            // one packed warp scan per round plus a carry.
            const uint32_t cw = ((n + kMatchThreads - 1) / kMatchThreads) * 32;
            const uint32_t wk0 = min(n, warp * cw), wk1 = min(n, wk0 + cw);
            // Stage the decoded LEN / OFF streams and the tag nibbles into shared memory with one round of
            // 16-byte async copies (sizes padded to 16 stay inside the slot areas / the record).
            {
                const uint32_t nl = (2 * n + 15) >> 4, no = (r.off_nbytes * n + 15) >> 4, nt = ((n + 1) / 2 + 15) >> 4;
                const uint8_t *gl = slot + sl.o_len, *go = slot + sl.o_off, *gt = r.rec + r.tags_off;
                for (uint32_t i = tid; i < nl; i += kMatchThreads) cp_async16(reinterpret_cast<uint8_t *>(s_len16) + 16 * i, gl + 16 * i);
                for (uint32_t i = tid; i < no; i += kMatchThreads) cp_async16(s_off + 16 * i, go + 16 * i);
                for (uint32_t i = tid; i < nt; i += kMatchThreads) cp_async16(s_tags + 16 * i, gt + 16 * i);
                cp_async_commit();
                if (tid == kMatchThreads - 1) s_wm = ld_acquire_u64(&ctl->watermark);   // it only grows; overlapped with the copies
                cp_async_wait_all();
                __syncthreads();
                TRACE_MARK(8);
            }
            const uint16_t *len16 = s_len16;
            const uint8_t *off_s = s_off;
            const uint16_t *extras = reinterpret_cast<const uint16_t *>(r.rec + r.extras_off);
            const uint8_t *tagsec = s_tags;
            const bool has_esc = r.n_extras != 0;                      // CTA-uniform
            // true (lit_len | match_len << 16) per sequence of a block with length escapes (rare): kept in the
            // slot's o_src area, which only the isolated path uses otherwise
            uint32_t *esc_val = reinterpret_cast<uint32_t *>(const_cast<uint8_t *>(slot) + sl.o_src);
            // A0 (only with escapes): escapes per warp -> extras base of each warp
            uint32_t esc_base = 0;
            if (has_esc) {
                uint32_t esc = 0;
                for (uint32_t k = wk0 + lane; k < wk1; k += 32) {
                    const uint32_t v = len16[k];
                    esc += ((v & 0xFFu) == 255) + ((v >> 8) == 255);
                }
                esc = __reduce_add_sync(0xFFFFFFFFu, esc);
                if (lane == 0) ws3[warp][0] = esc;
                __syncthreads();
                uint32_t tot = 0;
#pragma unroll
                for (uint32_t w = 0; w < kMatchWarps; w++) { const uint32_t x = ws3[w][0]; if (w < warp) esc_base += x; tot += x; }
                ok = tot == r.n_extras;
                __syncthreads();
            }
            // A: one packed warp scan per round. dm[k] receives the warp-relative exclusive prefix
            //    (literals before k | bytes before k << 16); the warp totals go to shared memory.
            uint32_t sum_ll = 0, sum_all = 0, any_esc = 0;
            if (ok) {
                uint32_t e_carry = esc_base, carry = 0;
                for (uint32_t kb = wk0; kb < wk1; kb += 32) {
                    const uint32_t k = kb + lane;
                    const bool act = k < wk1;
                    uint32_t ll = 0, ml = 0;
                    if (act) { const uint32_t v = len16[k]; ll = v & 0xFFu; ml = (v >> 8) + 4; }
                    const uint32_t e_ll = ll == 255, e_ml = ml == 259;
                    any_esc |= e_ll | e_ml;
                    if (has_esc) {
                        uint32_t etot;
                        uint32_t e = e_carry + warp_excl_scan(e_ll + e_ml, lane, etot);
                        if (e_ll) ll = extras[e++];
                        if (e_ml) ml = (uint32_t)extras[e] + 4;
                        e_carry += etot;
                        if (act) esc_val[k] = ll | ml << 16;            // true lengths for pass B
                    }
                    uint32_t ptot;
                    const uint32_t pre = warp_excl_scan(ll | (ll + ml) << 16, lane, ptot);
                    if (act) dm[k] = carry + pre;
                    carry += ptot;
                    sum_ll += ll;
                    sum_all += ll + ml;
                }
                sum_ll = __reduce_add_sync(0xFFFFFFFFu, sum_ll);
                sum_all = __reduce_add_sync(0xFFFFFFFFu, sum_all);
                any_esc = __reduce_or_sync(0xFFFFFFFFu, any_esc);
                if (lane == 0) { ws3[warp][0] = sum_ll; ws3[warp][1] = sum_all; ws3[warp][2] = any_esc; }
            }
            __syncthreads();
            TRACE_MARK(9);
            uint32_t ll_base = 0, all_base = 0, ll_total = 0, all_total = 0;
            if (ok) {
                uint32_t esc_seen = 0;
#pragma unroll
                for (uint32_t w = 0; w < kMatchWarps; w++) {
                    const uint32_t xa = ws3[w][0], xb = ws3[w][1];
                    if (w < warp) { ll_base += xa; all_base += xb; }
                    ll_total += xa; all_total += xb; esc_seen |= ws3[w][2];
                }
                ok = ll_total <= r.n_lit && all_total + (r.n_lit - ll_total) == blen && (has_esc || !esc_seen);
            }
            if (ok) {
                // B: elementwise. Every partial sum is <= block_len <= 16384 now, so st, d < 16384.
                const unsigned long long lit_a = (unsigned long long)__cvta_generic_to_global(slot + sl.o_lit);
                const unsigned long long out_a = (unsigned long long)__cvta_generic_to_global(out);
                const uint32_t onb = r.off_nbytes;                     // 1..8
                const uint64_t src_mask = ~0ull >> (64 - 8 * onb);
                const uint32_t blk32 = (uint32_t)blk;                  // n_blocks < 2^32 (checked by open)
                bool bad = false;
                uint32_t below = 0;                                    // 1 + highest earlier block read (upper bound)
                const uint32_t base = ll_base | all_base << 16;
                for (uint32_t kb = wk0; kb < wk1; kb += 32) {
                    const uint32_t k = kb + lane;
                    uint32_t tg = 0;
                    if (k < wk1) {
                        uint32_t ll, ml;
                        if (has_esc) { const uint32_t v = esc_val[k]; ll = v & 0xFFFFu; ml = v >> 16; }
                        else { const uint32_t v = len16[k]; ll = v & 0xFFu; ml = (v >> 8) + 4; }
                        const uint32_t pre = dm[k] + base;
                        const uint32_t lp = pre & 0xFFFFu;             // first literal of sequence k
                        const uint32_t st = pre >> 16;                 // in-block offset where sequence k starts
                        const uint32_t d = st + ll;                    // ... and where its match starts
                        // src = the onb bytes at off_s[k * onb]: three aligned words, funnel-shifted and masked
                        const uint32_t p = k * onb, sh = (p & 3u) * 8;
                        const uint32_t *wp = reinterpret_cast<const uint32_t *>(off_s + (p & ~3u));
                        const uint32_t w0 = wp[0], w1 = wp[1], w2 = wp[2];
                        const uint32_t lo = __funnelshift_r(w0, w1, sh), hi = __funnelshift_r(w1, w2, sh);
                        const uint64_t src = (((uint64_t)hi << 32) | lo) & src_mask;
                        tg = (tagsec[k >> 1] >> ((k & 1) * 4)) & 15u;
                        atomicOr(&bm2[st >> 5].x, 1u << (st & 31));
                        atomicOr(&bm2[d >> 5].y, 1u << (d & 31));
                        *reinterpret_cast<ulonglong2 *>(&delta[2 * k + 1]) = make_ulonglong2(lit_a + lp - st, out_a + src - d);
                        dm[k] = d | ml << 16;
                        if (src + ml > B0 + d) bad = true;             // strictly before, non-overlapping
                        // FORMAT.md section 4: tag 0 iff the source range lies entirely below the block
                        if ((tg == 0) != (src + ml <= B0)) bad = true;
                        // a source that starts in block sb < blk ends in block sb or sb + 1 (ml <= 16384)
                        const uint64_t sb = src >> kBlockLog2;
                        if (sb < blk) below = max(below, min((uint32_t)sb + 2u, blk32));
                    }
                    const uint32_t tm = __ballot_sync(0xFFFFFFFFu, tg != 0);
                    if (tm) {                                          // warp-aggregated append to the tag list
                        uint32_t tb = 0;
                        if (lane == 0) tb = atomicAdd(&s_ntag, (uint32_t)__popc(tm));
                        tb = __shfl_sync(0xFFFFFFFFu, tb, 0);
                        if (tg) {
                            tlist[tb + __popc(tm & lt)] = (uint16_t)(k | tg << 12);
                            atomicAdd(&s_cnt[tg], 1u);
                        }
                    }
                }
                if (tid == kMatchThreads - 1) {                        // trailing literals: run 2n+1
                    if (all_total < blen) atomicOr(&bm2[all_total >> 5].x, 1u << (all_total & 31));
                    delta[2 * n + 1] = lit_a + ll_total - all_total;
                }
                below = __reduce_max_sync(0xFFFFFFFFu, below);
                if (lane == 0 && below) atomicMax(&s_below, below);
                if (__any_sync(0xFFFFFFFFu, bad) && lane == 0) s_bad = 1;
            }
            __syncthreads();
            TRACE_MARK(1);
            ok = ok && !s_bad;
            if (!ok && tid == 0) raise(ctl, kStTokens, blk);
        }                                                              // (a bad record or stream was raised by k_entropy)
        if (ok) {
            // rk[w] = number of S and D bits in the words before w; tag list sorted by level
            {
                uint32_t p0 = 0, p1 = 0;
                if (tid < 256) {
                    const uint4 w = reinterpret_cast<const uint4 *>(bm2)[tid];        // words 2*tid, 2*tid+1
                    p0 = __popc(w.x) + __popc(w.y); p1 = __popc(w.z) + __popc(w.w);
                }
                uint32_t r0, d0, t0, t1;
                block_excl_scan2(p0 + p1, 0, ws2, r0, d0, t0, t1);
                if (tid < 256) reinterpret_cast<uint32_t *>(rk)[tid] = r0 | (r0 + p0) << 16;
            }
            const uint32_t ntag = s_ntag;
            const bool one_level = s_cnt[1] == ntag;                   // every tagged match has tag 1: no sorting
            const uint16_t *lst = tlist;
            if (!one_level) {
                __syncthreads();                                       // everybody has read s_cnt[1]
                if (tid == 0) {
                    uint32_t acc = 0;
                    for (int t = 0; t < 16; t++) { s_cur[t] = acc; acc += s_cnt[t]; s_cnt[t] = acc; }   // s_cnt[t] = end of level t
                }
                __syncthreads();
                for (uint32_t i = tid; i < ntag; i += kMatchThreads) {
                    const uint32_t e = tlist[i];
                    slist[atomicAdd(&s_cur[e >> 12], 1u)] = (uint16_t)e;
                }
                lst = slist;
            }
            // wait until every earlier block this block copies from is complete
            const uint64_t below = s_below;
            TRACE_MARK(2);
            if (warp == 0 && s_wm < below) wait_for_blocks(ctl, done, epoch, s_wm, below, true);
            __syncthreads();
            TRACE_MARK(3);
            // ---- pass 0: every output byte from delta[r(o)] + o; 16 byte loads in flight per thread
            const unsigned long long outB = (unsigned long long)__cvta_generic_to_global(out) + B0;
            uint32_t ob = 4 * tid;
            if (n == 0 && out_aligned4) {
                // a block without matches (incompressible data) is its literal stream: straight word copy
                const uint32_t *lw = reinterpret_cast<const uint32_t *>(slot + sl.o_lit);
                for (; ob + 12 * kMatchThreads + 4 <= blen; ob += 16 * kMatchThreads) {
                    const uint32_t i = ob >> 2;
                    const uint32_t a = lw[i], b = lw[i + kMatchThreads], c = lw[i + 2 * kMatchThreads], d = lw[i + 3 * kMatchThreads];
                    store4(outB + ob, a, 1u); store4(outB + ob + 4 * kMatchThreads, b, 1u);
                    store4(outB + ob + 8 * kMatchThreads, c, 1u); store4(outB + ob + 12 * kMatchThreads, d, 1u);
                }
            } else if (out_aligned4) {
                // word-granular gather (see plan_group): per step up to 4 aligned word loads, predicated on need
                for (; ob + (kWordUnroll - 1) * 4 * kMatchThreads + 4 <= blen; ob += kWordUnroll * 4 * kMatchThreads) {
                    GroupPlan g[kWordUnroll];
                    uint32_t alo[kWordUnroll], ahi[kWordUnroll], blo[kWordUnroll], bhi[kWordUnroll], v[kWordUnroll];
#pragma unroll
                    for (int u = 0; u < (int)kWordUnroll; u++) g[u] = plan_group(bm2, rk, delta, ob + u * 4 * kMatchThreads);
#pragma unroll
                    for (int u = 0; u < (int)kWordUnroll; u++) {
                        const unsigned long long wa = g[u].aA & ~3ull, wb = g[u].aB & ~3ull;
                        const uint32_t fa = (uint32_t)g[u].aA & 3u, fb = (uint32_t)g[u].aB & 3u, k = g[u].k;
                        // a multi-boundary group takes the per-byte path below: its aB belongs to a run that starts
                        // after byte k and may point up to 2 bytes before that run's source, i.e. before the buffer
                        const bool useB = k < 4 && !g[u].multi;
                        alo[u] = ldg_u32(wa);
                        ahi[u] = fa + k > 4 ? ldg_u32(wa + 4) : 0u;            // k = 4 for a group inside one run
                        blo[u] = useB ? ldg_u32(wb) : 0u;
                        bhi[u] = (useB && fb + (4 - k) > 4) ? ldg_u32(wb + 4) : 0u;
                    }
#pragma unroll
                    for (int u = 0; u < (int)kWordUnroll; u++) {
                        const uint32_t k = g[u].k;
                        const uint32_t va = __funnelshift_r(alo[u], ahi[u], 8 * ((uint32_t)g[u].aA & 3u));
                        const uint32_t vb = __funnelshift_r(blo[u], bhi[u], 8 * ((uint32_t)g[u].aB & 3u));
                        v[u] = k < 4 ? (va & ((1u << (8 * k)) - 1u)) | (vb << (8 * k)) : va;
                        if (g[u].multi) {                                      // two or more boundaries: byte by byte
                            const Addr4 a = run_addresses(bm2, rk, delta, ob + u * 4 * kMatchThreads);
                            v[u] = ldg_u8(a.a0) | ldg_u8(a.a1) << 8 | ldg_u8(a.a2) << 16 | ldg_u8(a.a3) << 24;
                        }
                    }
#pragma unroll
                    for (int u = 0; u < (int)kWordUnroll; u++) store4(outB + ob + u * 4 * kMatchThreads, v[u], 1u);
                }
            } else {
                for (; ob + 12 * kMatchThreads + 4 <= blen; ob += 16 * kMatchThreads) {
                    Addr4 a[4];
                    uint32_t b[4][4];
#pragma unroll
                    for (int u = 0; u < 4; u++) a[u] = run_addresses(bm2, rk, delta, ob + u * 4 * kMatchThreads);
#pragma unroll
                    for (int u = 0; u < 4; u++) {
                        b[u][0] = ldg_u8(a[u].a0); b[u][1] = ldg_u8(a[u].a1); b[u][2] = ldg_u8(a[u].a2); b[u][3] = ldg_u8(a[u].a3);
                    }
#pragma unroll
                    for (int u = 0; u < 4; u++)
                        store4(outB + ob + u * 4 * kMatchThreads, b[u][0] | b[u][1] << 8 | b[u][2] << 16 | b[u][3] << 24, 0u);
                }
            }
            for (; ob + 4 <= blen; ob += 4 * kMatchThreads) {
                const Addr4 a = run_addresses(bm2, rk, delta, ob);
                const uint32_t b0 = ldg_u8(a.a0), b1 = ldg_u8(a.a1), b2 = ldg_u8(a.a2), b3 = ldg_u8(a.a3);
                store4(outB + ob, b0 | b1 << 8 | b2 << 16 | b3 << 24, out_aligned4);
            }
            if (tid < (blen & 3u)) {                                   // ragged tail of a short last block
                const uint32_t o = (blen & ~3u) + tid;
                const uint2 w = bm2[o >> 5];
                const uint32_t m = (2u << (o & 31u)) - 1u;
                const uint32_t r0 = (uint32_t)rk[o >> 5] + __popc(w.x & m) + __popc(w.y & m);
                *reinterpret_cast<uint8_t *>(outB + o) = (uint8_t)ldg_u8(delta[r0] + o);
            }
            TRACE_MARK(4);
            // ---- matches whose source reaches into this block, level by level, 8 lanes per match
            if (ntag) {
                uint32_t i0 = 0;
                for (uint32_t level = 1; level < 16 && i0 < ntag; level++) {
                    const uint32_t i1 = one_level ? ntag : s_cnt[level];
                    if (i0 == i1) continue;                            // CTA-uniform
                    __syncthreads();                                   // the previous level (or pass 0) is in place
                    // 8 lanes per match, 4 matches per step: the first 16 bytes of each (2 per lane) are loaded
                    // before any is stored, so a step costs one round trip instead of four
                    const uint32_t l8 = tid & 7u, G = kMatchThreads / 8;
                    for (uint32_t ib = i0 + (tid >> 3); ib < i1; ib += 4 * G) {
                        unsigned long long sp[4], dp[4];
                        uint32_t ml[4], v0[4], v1[4];
#pragma unroll
                        for (int u = 0; u < 4; u++) {
                            const uint32_t i = ib + u * G;
                            ml[u] = 0; sp[u] = dp[u] = 0;
                            if (i < i1) {
                                const uint32_t k = lst[i] & 0xFFFu;
                                const uint32_t dmv = dm[k], d = dmv & 0xFFFFu;
                                ml[u] = dmv >> 16;
                                sp[u] = delta[2 * k + 2] + d; dp[u] = outB + d;
                            }
                        }
#pragma unroll
                        for (int u = 0; u < 4; u++) {
                            v0[u] = l8 < ml[u] ? ldg_u8(sp[u] + l8) : 0;
                            v1[u] = l8 + 8 < ml[u] ? ldg_u8(sp[u] + l8 + 8) : 0;
                        }
#pragma unroll
                        for (int u = 0; u < 4; u++) {
                            if (l8 < ml[u]) *reinterpret_cast<uint8_t *>(dp[u] + l8) = (uint8_t)v0[u];
                            if (l8 + 8 < ml[u]) *reinterpret_cast<uint8_t *>(dp[u] + l8 + 8) = (uint8_t)v1[u];
                        }
#pragma unroll
                        for (int u = 0; u < 4; u++) {                  // the rest of a long match, 4 loads in flight
                            for (uint32_t j = 16 + l8; j < ml[u]; j += 32) {
                                const uint32_t a = ldg_u8(sp[u] + j);
                                const uint32_t b = j + 8 < ml[u] ? ldg_u8(sp[u] + j + 8) : 0;
                                const uint32_t c = j + 16 < ml[u] ? ldg_u8(sp[u] + j + 16) : 0;
                                const uint32_t e = j + 24 < ml[u] ? ldg_u8(sp[u] + j + 24) : 0;
                                *reinterpret_cast<uint8_t *>(dp[u] + j) = (uint8_t)a;
                                if (j + 8 < ml[u]) *reinterpret_cast<uint8_t *>(dp[u] + j + 8) = (uint8_t)b;
                                if (j + 16 < ml[u]) *reinterpret_cast<uint8_t *>(dp[u] + j + 16) = (uint8_t)c;
                                if (j + 24 < ml[u]) *reinterpret_cast<uint8_t *>(dp[u] + j + 24) = (uint8_t)e;
                            }
                        }
                    }
                    i0 = i1;
                }
            }
        }
        // publish (also for a bad block: later blocks must not wait forever)
        __syncthreads();
        TRACE_MARK(5);
        if (tid == 0) st_release_u32(done + blk, epoch);
        TRACE_MARK(7);
    }
  }
    // last CTA out re-arms the ticket for the next launch
    if (tid == 0) {
        __threadfence();
        if (atomicAdd(&ctl->ticket_exit, 1u) == gridDim.x - 1) {
            ctl->ticket = 0;
            ctl->ticket_exit = 0;
            __threadfence();
        }
    }
}

}  // namespace aceapex
