// Match layer: token parse (FORMAT.md section 4), literal placement and absolute-offset copies
// (PAPER.md:19, :27), with cross-block ordering by ticket + watermark ("any block decodes once
// the blocks holding its source bytes are present").
#pragma once
#include "entropy.cuh"

namespace aceapex {

// Threads per match CTA: the parser-granularity knob of PAPER.md:86-92 (Table 3) in this design (one CTA
// cooperates on one 16 KiB block). Swept through -DACEAPEX_MATCH_THREADS (128, 256 or 512).
#ifndef ACEAPEX_MATCH_THREADS
#define ACEAPEX_MATCH_THREADS 256
#endif
constexpr uint32_t kMatchThreads = ACEAPEX_MATCH_THREADS;
constexpr uint32_t kMatchWarps = kMatchThreads / 32;
static_assert(kMatchThreads == 128 || kMatchThreads == 256 || kMatchThreads == 512, "match CTA size");

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
__device__ inline unsigned long long wait_for_blocks(Control *ctl, const uint32_t *done, uint32_t epoch,
                                                     unsigned long long w, unsigned long long below)
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
// Output-centric and branch-free. After the parse every output byte belongs to exactly one *run*: a
// non-empty literal run, a match, or the trailing literals. Runs are numbered in output order (empty
// literal runs get no number), so ONE bitmap over the 16,384 output offsets - bit o set iff a run starts
// at o - names the run that owns offset o as
//     r(o) = #bits <= o  -  1                      (a rank word + one popcount, no search)
// and its source byte sits at address delta[r] + o, where delta[r] is
//     literal run: &LIT[litpos] - start             (decoded LIT stream in the slot)
//     match:       &out[src]    - dst               (absolute offset into the output buffer)
// so literals and copies are the same instruction sequence (no staging tile for the gather: in-block
// sources are read back from the output buffer as well, which gives cross-block and in-block copies
// one address space).
//
// Matches with tag >= 1 (source range reaches into this block, FORMAT.md section 4) are produced
// by pass 0 with whatever the buffer held and then rewritten level by level from a list sorted by tag.

// Dynamic shared memory of one match CTA (bytes), for a slot capacity of ms sequences and offset width W:
//   cb    uint2 [kB / 32]   {run-start bits of 32 output offsets, number of run starts before them}
//   stage u8 [warps][512]   16-byte store staging, one 512-byte tile per warp
//   delta u64 [2 ms + 2]    per run (at most 2 n + 1)
//   dm    u32 [ms]          per sequence: dst | match_len << 16 (before the main pass: true lit_len | match_len << 16
//                           of a block with length escapes)
//   mrun  u16 [ms]          per sequence: run number of its match
//   tlist u16 [ms]          tagged matches, unsorted: the sequence number k (its tag is read again from the staged nibbles)
//   len   u16 [ms]          staged LEN stream; after the parse: tag list sorted by level
//   off   u8 [W ms + 16]    staged OFF stream (the word-wise offset read may touch 11 bytes past the last offset)
//   tags  u8 [pad16(ms/2)]  staged tag nibbles
constexpr uint32_t kCbWords = kB / 32;                              // 512 at 16 KiB
constexpr uint32_t kMatchFixedSmem = kCbWords * 8 + kMatchWarps * 512;

__host__ __device__ inline uint32_t match_smem_bytes(uint32_t ms, uint32_t W)
{
    return kMatchFixedSmem + (16 * ms + 16) + 4 * ms + 2 * ms + 2 * ms + 2 * ms + (W * ms + 16) + ((ms / 2 + 15u) & ~15u);
}

__device__ inline uint32_t ldg_u8(unsigned long long a)
{
    uint32_t v;
    asm volatile("ld.global.u8 %0, [%1];" : "=r"(v) : "l"(a) : "memory");
    return v;
}
__device__ inline uint32_t ldg_u32(unsigned long long a)
{
    uint32_t v;
    asm volatile("ld.global.u32 %0, [%1];" : "=r"(v) : "l"(a) : "memory");
    return v;
}
__device__ inline uint32_t shl_clamp(uint32_t v, uint32_t s)   // PTX shl: shift amounts >= 32 give 0
{
    uint32_t r;
    asm("shl.b32 %0, %1, %2;" : "=r"(r) : "r"(v), "r"(s));
    return r;
}

// ---- bulk async copies (TMA, sm_90+: cp.async.bulk, SASS UBLKCP) completing on a shared-memory mbarrier --------
// One thread posts the expected byte count and issues the copies; every thread then waits for the barrier's phase.
__device__ inline uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ inline void mbar_init(unsigned long long *bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ inline void mbar_expect_tx(unsigned long long *bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ inline void bulk_copy_g2s(void *dst_smem, const void *src, uint32_t bytes, unsigned long long *bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(dst_smem)), "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}
__device__ inline void mbar_wait(unsigned long long *bar, uint32_t parity)
{
    asm volatile("{\n"
                 ".reg .pred p;\n"
                 "MBAR_WAIT:\n"
                 "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
                 "@p bra MBAR_DONE;\n"
                 "bra MBAR_WAIT;\n"
                 "MBAR_DONE:\n"
                 "}" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}

// Exclusive prefix sum of one value per thread over the CTA.
__device__ inline uint32_t block_excl_scan(uint32_t a, uint32_t *ws /* [kMatchWarps] smem */)
{
    const uint32_t lane = lane_id(), warp = threadIdx.x >> 5;
    uint32_t wa;
    const uint32_t ia = warp_excl_scan(a, lane, wa);
    __syncthreads();
    if (lane == 0) ws[warp] = wa;
    __syncthreads();
    uint32_t ba = 0;
#pragma unroll
    for (uint32_t w = 0; w < kMatchWarps; w++) {
        const uint32_t xa = ws[w];
        if (w < warp) ba += xa;
    }
    return ba + ia;
}

// Run of output byte o (any o < block_len).
__device__ inline uint32_t run_of(const uint2 *cb, uint32_t o)
{
    const uint2 w = cb[o >> 5];
    return w.y + __popc(w.x & (0xFFFFFFFFu >> (31u - (o & 31u)))) - 1u;
}

// Output bytes o .. o+3 (o a multiple of 4), byte by byte: any number of run boundaries inside the group.
__device__ inline uint32_t gather_bytes(const uint2 *cb, const unsigned long long *delta, uint32_t o)
{
    const uint2 w = cb[o >> 5];
    const uint32_t sh = o & 31u;
    const uint32_t r0 = w.y + __popc(w.x & (0xFFFFFFFFu >> (31u - sh))) - 1u;
    const uint32_t t = w.x >> sh;
    const uint32_t r1 = r0 + ((t >> 1) & 1u), r2 = r1 + ((t >> 2) & 1u), r3 = r2 + ((t >> 3) & 1u);
    return ldg_u8(delta[r0] + o) | ldg_u8(delta[r1] + o + 1) << 8 | ldg_u8(delta[r2] + o + 2) << 16 | ldg_u8(delta[r3] + o + 3) << 24;
}

// Word-granular plan of output bytes o .. o+3: the run of byte 0 with the address aA that byte 0 maps to, the
// position k of the first run boundary inside the group (4 = none), the run after it with the address aB that
// BYTE 0 would map to in that run (its bytes k .. 3 are the ones taken) and whether there is a second boundary
// (then the group takes the per-byte path). With at most one boundary the four bytes are two (unaligned) 32-bit
// windows, each fetched as one or two ALIGNED words instead of four byte loads that touch the same cache lines
// four times. A word is only loaded if it holds at least one byte that is really taken, so no load ever leaves
// the buffer its run lives in.
struct GroupPlan { unsigned long long aA, aB; uint32_t k, multi; };
__device__ inline GroupPlan plan_group(const uint2 *cb, const unsigned long long *delta, uint32_t o)
{
    const uint2 w = cb[o >> 5];
    const uint32_t sh = o & 31u;
    const uint32_t rA = w.y + __popc(w.x & (0xFFFFFFFFu >> (31u - sh))) - 1u;
    const uint32_t x = (w.x >> sh) & 0xEu;
    GroupPlan g;
    g.k = (uint32_t)__ffs(x | 16u) - 1u;
    g.multi = x & (x - 1u);
    g.aA = delta[rA] + o;
    g.aB = delta[rA + __popc(x)] + o;
    return g;
}

struct GroupLoads { uint32_t alo, ahi, blo, bhi; };
__device__ inline GroupLoads load_group(const GroupPlan &g)
{
    const unsigned long long wa = g.aA & ~3ull, wb = g.aB & ~3ull;
    const uint32_t fa = (uint32_t)g.aA & 3u, fb = (uint32_t)g.aB & 3u, k = g.k;
    const bool useB = k < 4 && !g.multi;
    GroupLoads l;
    l.alo = ldg_u32(wa);                                               // byte 0 lives here
    l.ahi = fa + k > 4 ? ldg_u32(wa + 4) : 0u;                         // bytes up to k-1 reach the next word
    l.blo = (useB && fb + k < 4) ? ldg_u32(wb) : 0u;                   // byte k lives in the low word
    l.bhi = (useB && fb) ? ldg_u32(wb + 4) : 0u;                       // byte 3 lives in the high word
    return l;
}
__device__ inline uint32_t merge_group(const GroupPlan &g, const GroupLoads &l)
{
    const uint32_t va = __funnelshift_r(l.alo, l.ahi, 8 * ((uint32_t)g.aA & 3u));
    const uint32_t vb = __funnelshift_r(l.blo, l.bhi, 8 * ((uint32_t)g.aB & 3u));
    const uint32_t mk = shl_clamp(0xFFFFFFFFu, 8 * g.k);               // bytes k .. 3 (none for k = 4)
    return (va & ~mk) | (vb & mk);
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
__device__ inline void stg_v4(unsigned long long a, uint4 v)
{
    asm volatile("st.global.v4.u32 [%0], {%1, %2, %3, %4};" ::"l"(a), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
}

// kOutAlign: alignment of the output buffer (16, 4 or 1), a template parameter so that each instantiation carries one
// store path (measured on mixed_1g: k_match 2.20 -> 2.07 ms against the run-time switch).
template <uint32_t kOutAlign>
__global__ void __launch_bounds__(kMatchThreads) k_match(Container cv, SlotLayout sl, const uint8_t *slots,
                                                          uint64_t first, uint32_t count, uint8_t *out,
                                                          Control *ctl, uint32_t *done,
                                                          uint32_t epoch, uint64_t range_lo)
{
    extern __shared__ __align__(16) uint8_t smem[];
    __shared__ uint32_t ws4[kMatchWarps][4];
    __shared__ uint32_t ws1[kMatchWarps];
    __shared__ uint32_t s_ticket, s_ntag, s_bad;
    __shared__ unsigned long long s_wm, s_last;
    __shared__ uint32_t s_cnt[16], s_cur[16];
    __shared__ __align__(8) unsigned long long s_mbar;                 // completion of a block's staging copies

    const uint32_t ms = sl.ms;
    uint2 *cb = reinterpret_cast<uint2 *>(smem);                                    // [kCbWords]
    uint8_t *stage = smem + kCbWords * 8;                                                   // [kMatchWarps][512]
    unsigned long long *delta = reinterpret_cast<unsigned long long *>(smem + kMatchFixedSmem);   // [2*ms+2]
    uint32_t *dm = reinterpret_cast<uint32_t *>(smem + kMatchFixedSmem + 16 * ms + 16);           // [ms]
    uint16_t *mrun = reinterpret_cast<uint16_t *>(dm + ms);                         // [ms]
    uint16_t *tlist = mrun + ms;                                                    // [ms]
    uint16_t *s_len16 = tlist + ms;                                                 // [ms] staged LEN stream (u8 pairs)
    uint16_t *slist = s_len16;                                                      // [ms] tag list sorted by tag (after the parse)
    uint8_t *s_off = reinterpret_cast<uint8_t *>(s_len16 + ms);                     // [W*ms+16] staged OFF stream
    uint8_t *s_tags = s_off + cv.W * ms + 16;                                       // staged tag nibbles

    const uint32_t tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5;
    const uint32_t lt = (1u << lane) - 1u;
    constexpr uint32_t out_align = kOutAlign;
    constexpr uint32_t out_aligned4 = out_align >= 4;
    constexpr uint32_t kWordsPerThread = kCbWords >= kMatchThreads ? kCbWords / kMatchThreads : 1;   // rank scan
    static_assert(kCbWords % kWordsPerThread == 0, "bitmap words per thread");
    if (tid == 0) mbar_init(&s_mbar, 1);
    uint32_t stage_phase = 0;                                          // parity of the staging barrier's current phase
  // Persistent CTAs: each takes block after block from the ticket counter until none is left.
  for (;;) {
    __syncthreads();                                                   // the previous block's shared state is dead
    if (tid == 0) {
        s_ticket = atomicAdd(&ctl->ticket, 1u);
        s_last = 0;
        s_ntag = 0;
        s_bad = 0;
    }
    if (tid < 16) s_cnt[tid] = 0;
    for (uint32_t i = tid; i < kCbWords / 2; i += kMatchThreads) reinterpret_cast<uint4 *>(cb)[i] = make_uint4(0, 0, 0, 0);
    __syncthreads();
    if (s_ticket > count) break;                                       // tickets 1 .. count are blocks
    if (s_ticket == 0) {
        // Ticket 0 (a CTA that is certainly running) does not decode a block: it keeps the watermark moving
        // for everybody, kMatchThreads done flags per round trip, until this launch's blocks are done.
        const unsigned long long end = first + count;
        if (tid == 0) s_wm = ld_acquire_u64(&ctl->watermark);
        __syncthreads();
        unsigned long long w = s_wm;
        while (w < end) {
            const unsigned long long idx = w + tid;
            const bool f = idx >= end || ld_acquire_u32(done + idx) == epoch;
            const uint32_t m = __ballot_sync(0xFFFFFFFFu, f);
            if (lane == 0) ws1[warp] = m == 0xFFFFFFFFu ? 32u : (uint32_t)__ffs(~m) - 1u;
            __syncthreads();
            uint32_t lead = 0;
#pragma unroll
            for (uint32_t i = 0; i < kMatchWarps; i++) {
                const uint32_t c = ws1[i];
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
        if (ok) {
            // ---- parse (FORMAT.md section 4). Warp w owns the sequences [w*cw, (w+1)*cw), lane-strided:
            // in round i lane l holds sequence w*cw + 32*i + l, so loads coalesce and the prefix sums are
            // one packed warp scan per round plus a carry.
            const uint32_t cw = ((n + kMatchThreads - 1) / kMatchThreads) * 32;
            const uint32_t wk0 = min(n, warp * cw), wk1 = min(n, wk0 + cw);
            // Stage the decoded LEN / OFF streams and the tag nibbles into shared memory: three bulk async copies
            // (TMA: one instruction per stream, issued by one thread, completing on a shared-memory mbarrier; the
            // sizes padded to 16 stay inside the slot areas / the record) instead of a cp.async loop over all threads.
            if (n) {
                const uint32_t nl = (2 * n + 15) & ~15u, no = (r.off_nbytes * n + 15) & ~15u, nt = ((n + 1) / 2 + 15) & ~15u;
                if (tid == 0) {
                    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // the previous block's reads of these buffers are done (loop-top barrier)
                    mbar_expect_tx(&s_mbar, nl + no + nt);
                    bulk_copy_g2s(s_len16, slot + sl.o_len, nl, &s_mbar);
                    bulk_copy_g2s(s_off, slot + sl.o_off, no, &s_mbar);
                    bulk_copy_g2s(s_tags, r.rec + r.tags_off, nt, &s_mbar);
                }
                if (tid == kMatchThreads - 1) s_wm = ld_acquire_u64(&ctl->watermark);   // it only grows; overlapped with the copies
                if (warp == 0) mbar_wait(&s_mbar, stage_phase);       // one warp polls; the others sleep in the CTA barrier
                stage_phase ^= 1u;
                __syncthreads();                                       // (also publishes s_wm)
            } else {
                if (tid == kMatchThreads - 1) s_wm = ld_acquire_u64(&ctl->watermark);
                __syncthreads();
            }
            const uint16_t *len16 = s_len16;
            const bool has_esc = r.n_extras != 0;                      // CTA-uniform
            // E (only with length escapes): the true lit_len | match_len << 16 of every sequence goes to dm[k]
            if (has_esc) {
                const uint16_t *extras = reinterpret_cast<const uint16_t *>(r.rec + r.extras_off);
                uint32_t esc = 0;
                for (uint32_t k = wk0 + lane; k < wk1; k += 32) {
                    const uint32_t v = len16[k];
                    esc += ((v & 0xFFu) == 255) + ((v >> 8) == 255);
                }
                esc = __reduce_add_sync(0xFFFFFFFFu, esc);
                if (lane == 0) ws4[warp][0] = esc;
                __syncthreads();
                uint32_t e_carry = 0, tot = 0;
#pragma unroll
                for (uint32_t w = 0; w < kMatchWarps; w++) { const uint32_t x = ws4[w][0]; if (w < warp) e_carry += x; tot += x; }
                ok = tot == r.n_extras;                                // bounds every extras index below
                bool bad = false;
                if (ok)
                    for (uint32_t kb = wk0; kb < wk1; kb += 32) {
                        const uint32_t k = kb + lane;
                        const bool act = k < wk1;
                        const uint32_t v = act ? len16[k] : 0u;
                        uint32_t ll = v & 0xFFu, m4 = v >> 8;
                        const bool e_ll = ll == 255, e_ml = m4 == 255;
                        const uint32_t mA = __ballot_sync(0xFFFFFFFFu, e_ll), mB = __ballot_sync(0xFFFFFFFFu, e_ml);
                        const uint32_t e = e_carry + __popc(mA & lt) + __popc(mB & lt);   // order: sequence, literal before match
                        if (e_ll) ll = extras[e];
                        if (e_ml) m4 = extras[e + (e_ll ? 1u : 0u)];
                        e_carry += __popc(mA) + __popc(mB);
                        if (ll > kB || m4 + 4 > kB) bad = true;        // keeps every later sum inside 32 bits and both fields inside 16
                        if (act) dm[k] = ll | (m4 + 4) << 16;
                    }
                if (__any_sync(0xFFFFFFFFu, bad) && lane == 0) s_bad = 1;
                __syncthreads();                                       // (also: ws4 is reused below)
                ok = ok && !s_bad;
            }
            // A: per-warp sums of literal lengths, of all lengths and of non-empty literal runs
            uint32_t ll_base = 0, all_base = 0, ne_base = 0, ll_total = 0, all_total = 0, ne_total = 0;
            {
                uint32_t s_ll = 0, s_all = 0, s_ne = 0, esc_seen = 0;
                if (ok)
                    for (uint32_t k = wk0 + lane; k < wk1; k += 32) {
                        uint32_t ll, ml;
                        if (has_esc) { const uint32_t v = dm[k]; ll = v & 0xFFFFu; ml = v >> 16; }
                        else { const uint32_t v = len16[k]; ll = v & 0xFFu; ml = (v >> 8) + 4; esc_seen |= (ll == 255) | (ml == 259); }
                        s_ll += ll; s_all += ll + ml; s_ne += ll != 0;
                    }
                s_ll = __reduce_add_sync(0xFFFFFFFFu, s_ll);
                s_all = __reduce_add_sync(0xFFFFFFFFu, s_all);
                s_ne = __reduce_add_sync(0xFFFFFFFFu, s_ne);
                esc_seen = __reduce_or_sync(0xFFFFFFFFu, esc_seen);
                if (lane == 0) { ws4[warp][0] = s_ll; ws4[warp][1] = s_all; ws4[warp][2] = s_ne; ws4[warp][3] = esc_seen; }
                __syncthreads();
                uint32_t any_esc = 0;
#pragma unroll
                for (uint32_t w = 0; w < kMatchWarps; w++) {
                    const uint32_t xa = ws4[w][0], xb = ws4[w][1], xc = ws4[w][2];
                    if (w < warp) { ll_base += xa; all_base += xb; ne_base += xc; }
                    ll_total += xa; all_total += xb; ne_total += xc; any_esc |= ws4[w][3];
                }
                // an escape byte without an extras entry is invalid; the sums must tile the block exactly
                ok = ok && !any_esc && ll_total <= r.n_lit && all_total + (r.n_lit - ll_total) == blen;
            }
            if (ok) {
                // B: one packed warp scan per round. Every partial sum is <= block_len <= 16384 now, so both
                // 16-bit fields hold, every match start is < block_len and every run-start bit lands in cb.
                const unsigned long long lit_a = (unsigned long long)__cvta_generic_to_global(slot + sl.o_lit);
                const unsigned long long out_a = (unsigned long long)__cvta_generic_to_global(out);
                const uint32_t onb = r.off_nbytes;                     // 1..8
                const uint64_t src_mask = ~0ull >> (64 - 8 * onb);
                const uint8_t *off_s = s_off;
                bool bad = false;
                unsigned long long last = 0;                           // 1 + highest source byte below this block
                uint32_t carry = ll_base | all_base << 16, ne_carry = ne_base;
                for (uint32_t kb = wk0; kb < wk1; kb += 32) {
                    const uint32_t k = kb + lane;
                    const bool act = k < wk1;
                    uint32_t ll = 0, ml = 0;
                    if (act) {
                        if (has_esc) { const uint32_t v = dm[k]; ll = v & 0xFFFFu; ml = v >> 16; }
                        else { const uint32_t v = len16[k]; ll = v & 0xFFu; ml = (v >> 8) + 4; }
                    }
                    uint32_t ptot;
                    const uint32_t pre = carry + warp_excl_scan(ll | (ll + ml) << 16, lane, ptot);
                    carry += ptot;
                    const uint32_t nem = __ballot_sync(0xFFFFFFFFu, ll != 0);
                    const uint32_t rl = k + ne_carry + __popc(nem & lt);       // run number of the literal run (if any)
                    ne_carry += __popc(nem);
                    uint32_t tg = 0;
                    if (act) {
                        const uint32_t lp = pre & 0xFFFFu;             // first literal of sequence k
                        const uint32_t st = pre >> 16;                 // in-block offset where sequence k starts
                        const uint32_t d = st + ll;                    // ... and where its match starts
                        const uint32_t rm = rl + (ll != 0);            // run number of the match
                        // src = the onb bytes at off_s[k * onb]: aligned words, funnel-shifted and masked
                        const uint32_t p = k * onb, sh = (p & 3u) * 8;
                        const uint32_t *wp = reinterpret_cast<const uint32_t *>(off_s + (p & ~3u));
                        uint64_t src;
                        if (onb <= 4) {                                // CTA-uniform
                            src = __funnelshift_r(wp[0], wp[1], sh) & (uint32_t)src_mask;
                        } else {
                            const uint32_t w0 = wp[0], w1 = wp[1], w2 = wp[2];
                            src = (((uint64_t)__funnelshift_r(w1, w2, sh) << 32) | __funnelshift_r(w0, w1, sh)) & src_mask;
                        }
                        tg = (s_tags[k >> 1] >> ((k & 1) * 4)) & 15u;
                        // run-start bits: the literal run (if any) and the match
                        const uint32_t bS = ll ? 1u << (st & 31) : 0u, bD = 1u << (d & 31);
                        if ((st >> 5) == (d >> 5)) {
                            atomicOr(&cb[d >> 5].x, bS | bD);
                        } else {
                            atomicOr(&cb[st >> 5].x, bS);              // ll != 0 here
                            atomicOr(&cb[d >> 5].x, bD);
                        }
                        if (ll) delta[rl] = lit_a + lp - st;
                        // Range decode: a source below the range is not in the buffer; the isolated
                        // chase has already put this match's bytes in place, so the run copies itself onto itself.
                        const bool ext = src < range_lo;
                        delta[rm] = ext ? out_a + B0 : out_a + src - d;
                        dm[k] = d | ml << 16;
                        mrun[k] = (uint16_t)rm;
                        const uint64_t se = src + ml;
                        if (se > B0 + d) bad = true;                   // strictly before, non-overlapping
                        // FORMAT.md section 4: tag 0 iff the source range lies entirely below the block
                        if ((tg == 0) != (se <= B0)) bad = true;
                        if (!ext && src < B0) last = max(last, min((unsigned long long)se, (unsigned long long)B0));
                    }
                    const uint32_t tm = __ballot_sync(0xFFFFFFFFu, tg != 0);
                    if (tm) {                                          // warp-aggregated append to the tag list
                        uint32_t tb = 0;
                        if (lane == 0) tb = atomicAdd(&s_ntag, (uint32_t)__popc(tm));
                        tb = __shfl_sync(0xFFFFFFFFu, tb, 0);
                        if (tg) {
                            tlist[tb + __popc(tm & lt)] = (uint16_t)k;
                            atomicAdd(&s_cnt[tg], 1u);
                        }
                    }
                }
                if (tid == kMatchThreads - 1 && all_total < blen) {    // trailing literals: the last run
                    atomicOr(&cb[all_total >> 5].x, 1u << (all_total & 31));
                    delta[n + ne_total] = lit_a + ll_total - all_total;
                }
                {   // 64-bit warp maximum of `last`
                    const uint32_t hi = __reduce_max_sync(0xFFFFFFFFu, (uint32_t)(last >> 32));
                    const uint32_t lo = __reduce_max_sync(0xFFFFFFFFu, (uint32_t)(last >> 32) == hi ? (uint32_t)last : 0u);
                    if (lane == 0 && (hi | lo)) atomicMax(&s_last, (unsigned long long)hi << 32 | lo);
                }
                if (__any_sync(0xFFFFFFFFu, bad) && lane == 0) s_bad = 1;
            }
            __syncthreads();
            ok = ok && !s_bad;
            if (!ok && tid == 0) raise(ctl, kStTokens, blk);
        }                                                              // (a bad record or stream was raised by k_entropy)
        if (ok) {
            // cb[w].y = number of run starts in the words before w; tag list sorted by level
            {
                uint32_t p[kWordsPerThread], tot = 0;
                const bool mine = kWordsPerThread * tid < kCbWords;    // (a 4 KiB block has fewer words than threads)
#pragma unroll
                for (uint32_t i = 0; i < kWordsPerThread; i++) { p[i] = mine ? __popc(cb[kWordsPerThread * tid + i].x) : 0u; tot += p[i]; }
                uint32_t r0 = block_excl_scan(tot, ws1);
#pragma unroll
                for (uint32_t i = 0; i < kWordsPerThread; i++) { if (mine) cb[kWordsPerThread * tid + i].y = r0; r0 += p[i]; }
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
                    const uint32_t k = tlist[i];
                    slist[atomicAdd(&s_cur[(s_tags[k >> 1] >> ((k & 1) * 4)) & 15u], 1u)] = (uint16_t)k;
                }
                lst = slist;
            }
            // wait until every earlier block this block copies from is complete
            const uint64_t below = (s_last + kB - 1) >> kBlockLog2;    // number of leading blocks that must be complete
            if (warp == 0 && s_wm < below) wait_for_blocks(ctl, done, epoch, s_wm, below);
            __syncthreads();
            // ---- pass 0: every output byte from delta[r(o)] + o
            const unsigned long long outB = (unsigned long long)__cvta_generic_to_global(out) + B0;
            uint32_t ob = 0;                                           // first byte not produced by the tile loops
            if (n == 0 && out_align >= 16) {
                // a block without matches (incompressible data) is its literal stream: straight 16-byte copy
                const uint4 *lw = reinterpret_cast<const uint4 *>(slot + sl.o_lit);
                const uint32_t nv = blen >> 4;
                uint32_t i = tid;
                for (; i + 3 * kMatchThreads < nv; i += 4 * kMatchThreads) {
                    const uint4 a = lw[i], b = lw[i + kMatchThreads], c = lw[i + 2 * kMatchThreads], d = lw[i + 3 * kMatchThreads];
                    stg_v4(outB + 16 * i, a); stg_v4(outB + 16 * (i + kMatchThreads), b);
                    stg_v4(outB + 16 * (i + 2 * kMatchThreads), c); stg_v4(outB + 16 * (i + 3 * kMatchThreads), d);
                }
                for (; i < nv; i += kMatchThreads) stg_v4(outB + 16 * i, lw[i]);
                ob = nv << 4;
            } else if (out_aligned4) {
                // Word-granular gather (see plan_group). A warp takes 512-byte tiles: four steps of 128 consecutive
                // bytes (one word per lane, so the gathers of a step stay coalesced per run), all loads of the tile in
                // flight together; the four words of a lane are exchanged through the warp's staging tile so that the
                // output leaves as one 16-byte store per lane.
                uint8_t *stg = stage + warp * 512;
                const uint32_t n_tiles = blen >> 9;
                for (uint32_t t = warp; t < n_tiles; t += kMatchWarps) {
                    const uint32_t base = t << 9;
                    GroupPlan g[4];
                    GroupLoads l[4];
#pragma unroll
                    for (int u = 0; u < 4; u++) g[u] = plan_group(cb, delta, base + 128 * u + 4 * lane);
#pragma unroll
                    for (int u = 0; u < 4; u++) l[u] = load_group(g[u]);
#pragma unroll
                    for (int u = 0; u < 4; u++) {
                        uint32_t v = merge_group(g[u], l[u]);
                        if (g[u].multi) v = gather_bytes(cb, delta, base + 128 * u + 4 * lane);   // two or more boundaries
                        if (out_align >= 16) *reinterpret_cast<uint32_t *>(stg + 128 * u + 4 * lane) = v;
                        else store4(outB + base + 128 * u + 4 * lane, v, 1u);
                    }
                    if (out_align >= 16) {
                        __syncwarp();
                        const uint4 q = *reinterpret_cast<const uint4 *>(stg + 16 * lane);
                        stg_v4(outB + base + 16 * lane, q);
                        __syncwarp();                                  // the tile is rewritten by the next iteration
                    }
                }
                ob = n_tiles << 9;
            }
            // the rest (a short last block, an unaligned buffer): 4 bytes per thread, byte by byte
            for (uint32_t o = ob + 4 * tid; o + 4 <= blen; o += 4 * kMatchThreads)
                store4(outB + o, gather_bytes(cb, delta, o), out_aligned4);
            if (tid < (blen & 3u)) {                                   // ragged tail
                const uint32_t o = (blen & ~3u) + tid;
                *reinterpret_cast<uint8_t *>(outB + o) = (uint8_t)ldg_u8(delta[run_of(cb, o)] + o);
            }
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
                                const uint32_t k = lst[i];
                                const uint32_t dmv = dm[k], d = dmv & 0xFFFFu;
                                ml[u] = dmv >> 16;
                                sp[u] = delta[mrun[k]] + d; dp[u] = outB + d;
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
        if (tid == 0) st_release_u32(done + blk, epoch);
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
