// Entropy layer: 32-lane interleaved rANS decode of one token stream of one block by one warp
// (FORMAT.md section 3; PAPER.md:33 per-block ANS, :124 ref [6] interleaved rANS).
//
// Warp-parallel form of the sequential decoder: in round r lane l decodes symbol 32r + l; the
// lanes whose state fell below 2^16 take consecutive 16-bit words in lane order (ballot + popc),
// which is exactly the order in which the sequential decoder, visiting lanes 0..31 inside a
// round, would have consumed them.
#pragma once
#include "format.cuh"

namespace aceapex {

// Shared memory of the entropy decoder, per warp (bytes):
//   t8   [4096]  slot -> index of the present symbol that owns the slot. All t8 tables of a CTA sit in
//                one 4096-aligned region of the shared window, so a lookup address is
//                (x & 4095) | t8_base: one LOP3.
//   syml [256]   u64 per present symbol: lo = sym | (-c) << 8 (two's complement, 24 bit), hi = f
//   ring [512]   table build: 4096-bit symbol-start bitmap; decode: ring of 256 16-bit rANS words,
//                refilled with cp.async. (The build's 256-byte rank array borrows the tail of t8.)
constexpr uint32_t kT8Bytes = kM;
constexpr uint32_t kSymlBytes = 256 * 8;
constexpr uint32_t kRingBytes = 512;
// Warps per entropy CTA (each warp decodes one stream at a time with its own tables). Swept through
// -DACEAPEX_ENTROPY_WARPS (8 or 16; PAPER.md:86-92 sweeps the threads per parser the same way).
#ifndef ACEAPEX_ENTROPY_WARPS
#define ACEAPEX_ENTROPY_WARPS 16
#endif
constexpr uint32_t kEntropyWarps = ACEAPEX_ENTROPY_WARPS;
static_assert(kEntropyWarps == 4 || kEntropyWarps == 8 || kEntropyWarps == 16, "entropy CTA size");
constexpr uint32_t kEntropySmem = kEntropyWarps * (kT8Bytes + kSymlBytes + kRingBytes) + kT8Bytes;   // + alignment slack
constexpr uint32_t kRingWords = 256, kRingChunk = 64;

// Where one warp's tables live: generic pointers for the build, shared-window addresses for the loop.
struct WarpSmem {
    uint8_t *t8; uint2 *syml; uint8_t *ring;
    uint32_t a_t8, a_syml, a_ring;
};

__device__ inline uint32_t lds_u8(uint32_t a)
{
    uint32_t v;
    asm volatile("ld.shared.u8 %0, [%1];" : "=r"(v) : "r"(a));
    return v;
}
__device__ inline uint32_t lds_u16(uint32_t a)
{
    uint32_t v;
    asm volatile("ld.shared.u16 %0, [%1];" : "=r"(v) : "r"(a));
    return v;
}
__device__ inline uint2 lds_v2(uint32_t a)
{
    uint2 v;
    asm volatile("ld.shared.v2.u32 {%0, %1}, [%2];" : "=r"(v.x), "=r"(v.y) : "r"(a));
    return v;
}

__device__ inline uint32_t lane_id() { return threadIdx.x & 31u; }

// "Am I lane 0", read afresh every time. A leader branch written as `lane == 0` invites the compiler to thread
// several such tests into one and to duplicate the code between them for the two outcomes: lane 0 then runs
// its own copy of a whole stream decode beside the other 31 lanes (measured on k_entropy: 75 -> 180 us when one
// more leader branch was added to decode_unit). An opaque read keeps every leader branch a small diamond.
__device__ inline bool leader()
{
    uint32_t l;
    asm volatile("mov.u32 %0, %%laneid;" : "=r"(l));
    return l == 0;
}

__device__ inline uint32_t warp_excl_scan(uint32_t v, uint32_t lane, uint32_t &total)
{
    uint32_t inc = v;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        uint32_t t = __shfl_up_sync(0xFFFFFFFFu, inc, d);
        if (lane >= (uint32_t)d) inc += t;
    }
    total = __shfl_sync(0xFFFFFFFFu, inc, 31);
    return inc - v;
}

__device__ inline void cp_async4(void *smem_dst, const void *gsrc)
{
    const uint32_t d = (uint32_t)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(d), "l"(gsrc) : "memory");
}
__device__ inline void cp_async16(void *smem_dst, const void *gsrc)
{
    const uint32_t d = (uint32_t)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(d), "l"(gsrc) : "memory");
}
__device__ inline void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ inline void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }

// Build the two-level decode table of one stream in shared memory (FORMAT.md section 3 "Table").
// Returns false (warp-uniform) if the table section is invalid.
__device__ inline bool build_table(const uint8_t *tbl_sec, uint32_t tbl_bytes, uint8_t *t8, uint2 *syml,
                                   uint32_t *bmw /* [128] */, uint16_t *rk /* [128], may alias t8[3840..] */,
                                   uint32_t lane)
{
    if (tbl_bytes < 32) return false;
    const uint32_t bm = tbl_sec[lane];                   // presence of symbols 8*lane .. 8*lane+7
    uint32_t n_present;
    const uint32_t first = warp_excl_scan(__popc(bm), lane, n_present);
    if (n_present == 0 || tbl_bytes != 32 + 2 * n_present) return false;
    const uint16_t *fq = reinterpret_cast<const uint16_t *>(tbl_sec + 32);
    uint32_t f[8], sum = 0;
    bool bad = false;
    {
        uint32_t j = first;
#pragma unroll
        for (int k = 0; k < 8; k++) {
            f[k] = 0;
            if (bm >> k & 1u) {
                f[k] = fq[j++];
                if (f[k] < 1 || f[k] > kM) bad = true;
                sum += f[k];
            }
        }
    }
    if (__any_sync(0xFFFFFFFFu, bad)) return false;      // bounds every f before the scan
    uint32_t total;
    uint32_t c = warp_excl_scan(sum, lane, total);
    if (total != kM) return false;
    reinterpret_cast<uint4 *>(bmw)[lane] = make_uint4(0, 0, 0, 0);
    __syncwarp();
    {
        uint32_t j = first;
#pragma unroll
        for (int k = 0; k < 8; k++)
            if (bm >> k & 1u) {
                syml[j++] = make_uint2((8 * lane + k) | (0u - c) << 8, f[k]);   // c <= 4095
                atomicOr(&bmw[c >> 5], 1u << (c & 31));                          // symbol starts at slot c
                c += f[k];
            }
    }
    __syncwarp();
    {   // rank of each bitmap word = number of symbol starts in the words before it
        const uint4 w = reinterpret_cast<const uint4 *>(bmw)[lane];
        const uint32_t p0 = __popc(w.x), p1 = __popc(w.y), p2 = __popc(w.z), p3 = __popc(w.w);
        uint32_t tot;
        const uint32_t r0 = warp_excl_scan(p0 + p1 + p2 + p3, lane, tot);
        reinterpret_cast<uint2 *>(rk)[lane] = make_uint2(r0 | (r0 + p0) << 16, (r0 + p0 + p1) | (r0 + p0 + p1 + p2) << 16);
    }
    __syncwarp();
    // fill: per iteration the warp writes 512 slots, 16 consecutive bytes per lane
#pragma unroll 2
    for (uint32_t it = 0; it < 8; it++) {
        const uint32_t wi = 16 * it + (lane >> 1), h = (lane & 1u) * 16;
        const uint32_t w = bmw[wi];
        const uint32_t bits = (w >> h) & 0xFFFFu;
        // index of the symbol that owns the slot just before this lane's first slot
        uint32_t base = (uint32_t)rk[wi] + __popc(w & ((1u << h) - 1u)) - 1u;
        __syncwarp();                                    // rk borrows the tail of t8: read before the last write
        uint32_t o[4];
#pragma unroll
        for (int g = 0; g < 4; g++) {
            const uint32_t nib = (bits >> (4 * g)) & 0xFu;
            const uint32_t spread = (nib * 0x00204081u) & 0x01010101u;   // bit k -> byte k
            o[g] = spread * 0x01010101u + base * 0x01010101u;            // running symbol index per slot
            base = o[g] >> 24;
        }
        reinterpret_cast<uint4 *>(t8)[32 * it + lane] = make_uint4(o[0], o[1], o[2], o[3]);
    }
    __syncwarp();
    return true;
}

// One rANS round of the warp (FORMAT.md section 3), branch-free: decode this lane's symbol, then the
// lanes whose state fell below 2^16 take consecutive words in lane order. wpos2 = 2 * words consumed.
#define ACEAPEX_RANS_ROUND(SYM)                                                                        \
    {                                                                                                  \
        const uint32_t slot_ = x & (kM - 1);                                                           \
        const uint32_t i_ = lds_u8(slot_ | ws.a_t8);                                                   \
        const uint2 e_ = lds_v2(i_ * 8u + ws.a_syml);                                                  \
        x = e_.y * (x >> kProbBits) + (slot_ + (uint32_t)((int32_t)e_.x >> 8));                        \
        const bool need_ = x < kRansL;                                                                 \
        const uint32_t mask_ = __ballot_sync(0xFFFFFFFFu, need_);                                      \
        const uint32_t w_ = lds_u16(((wpos2 + 2u * __popc(mask_ & lt)) & (2 * kRingWords - 1)) | ws.a_ring); \
        if (need_) x = (x << 16) | w_;                                                                 \
        wpos2 += 2u * __popc(mask_);                                                                   \
        SYM = e_.x;                                                                                    \
    }

// Decode one stream (n symbols, n_words 16-bit words) into out[0, n). One warp. Returns true
// (warp-uniform) on success; false if the table or the rANS end conditions are violated (then
// out is unspecified but never written beyond n). A stream that consumes more words than it has
// reads stale ring entries (shared memory, in bounds) and fails the final word-count check.
__device__ inline bool decode_stream(uint32_t x /* this lane's initial state */, uint32_t n, uint32_t n_words,
                                     const uint8_t *tbl_sec, uint32_t tbl_bytes, const uint8_t *words_sec,
                                     uint8_t *out, const WarpSmem &ws, uint32_t lane)
{
    if (n == 0) return __all_sync(0xFFFFFFFFu, x == kRansL) && n_words == 0;
    __syncwarp();
    if (!build_table(tbl_sec, tbl_bytes, ws.t8, ws.syml, reinterpret_cast<uint32_t *>(ws.ring),
                     reinterpret_cast<uint16_t *>(ws.t8 + kT8Bytes - 256), lane))
        return false;
    // word ring: 4 chunks of 64 words; chunk k lives at ring[(k & 3) * 64 ...]
    const uint32_t wbytes = 2 * n_words;
    if (16 * lane < wbytes) cp_async16(ws.ring + 16 * lane, words_sec + 16 * lane);   // words 0 .. 255
    cp_async_commit();
    cp_async_wait_all();
    __syncwarp();
    const uint32_t lt = (1u << lane) - 1u;
    uint32_t wpos2 = 0, trigger2 = 2 * kRingChunk;
    uint8_t *op = out + lane;
    uint32_t rd = n >> 5;
    // Refill: when the words of chunk j are consumed, chunk j+4 is requested into its place; the wait
    // at the next firing has had >= 64 words of decoding to hide behind. Checked every 4 rounds
    // (<= 128 words): with firings up to j-1 done, chunks up to j+2 have landed, which covers
    // every word below trigger_j + 128 that the next 4 rounds can read.
#define ACEAPEX_RING_REFILL()                                                                          \
    while (wpos2 >= trigger2) {                                                                        \
        cp_async_wait_all();                                                                           \
        __syncwarp();                                                                                  \
        const uint32_t boff_ = trigger2 + 6 * kRingChunk + 4 * lane;   /* chunk trigger/64 + 3 */      \
        if (boff_ < wbytes) cp_async4(ws.ring + (boff_ & (2 * kRingWords - 1)), words_sec + boff_);   \
        cp_async_commit();                                                                             \
        trigger2 += 2 * kRingChunk;                                                                    \
    }
    for (; rd >= 4; rd -= 4) {
        ACEAPEX_RING_REFILL();
        uint32_t s0, s1, s2, s3;
        ACEAPEX_RANS_ROUND(s0);
        ACEAPEX_RANS_ROUND(s1);
        ACEAPEX_RANS_ROUND(s2);
        ACEAPEX_RANS_ROUND(s3);
        op[0] = (uint8_t)s0;
        op[32] = (uint8_t)s1;
        op[64] = (uint8_t)s2;
        op[96] = (uint8_t)s3;
        op += 128;
    }
    ACEAPEX_RING_REFILL();
    for (; rd; rd--) {
        uint32_t s0;
        ACEAPEX_RANS_ROUND(s0);
        op[0] = (uint8_t)s0;
        op += 32;
    }
    if (n & 31u) {                                                   // ragged last round
        ACEAPEX_RING_REFILL();
        const bool active = lane < (n & 31u);
        const uint32_t x_keep = x;
        uint32_t s0;
        {
            const uint32_t slot_ = x & (kM - 1);
            const uint32_t i_ = lds_u8(slot_ | ws.a_t8);
            const uint2 e_ = lds_v2(i_ * 8u + ws.a_syml);
            x = e_.y * (x >> kProbBits) + (slot_ + (uint32_t)((int32_t)e_.x >> 8));
            const bool need_ = active && x < kRansL;
            const uint32_t mask_ = __ballot_sync(0xFFFFFFFFu, need_);
            const uint32_t w_ = lds_u16(((wpos2 + 2u * __popc(mask_ & lt)) & (2 * kRingWords - 1)) | ws.a_ring);
            if (need_) x = (x << 16) | w_;
            wpos2 += 2u * __popc(mask_);
            s0 = e_.x;
        }
        if (active) op[0] = (uint8_t)s0; else x = x_keep;
    }
#undef ACEAPEX_RING_REFILL
    cp_async_wait_all();
    return __all_sync(0xFFFFFFFFu, x == kRansL) && wpos2 == wbytes;
}

// A RAW stream (FORMAT.md section 2, mode 1): the symbols are stored verbatim in the words
// section. Both ends are 16-byte aligned and padded inside their areas, so the warp copies whole uint4s.
// The unused rANS states must be 2^16 and the pad byte of an odd-length stream 0.
__device__ inline bool copy_raw_stream(uint32_t x, uint32_t n, const uint8_t *words_sec, uint8_t *out, uint32_t lane)
{
    bool ok = x == kRansL;
    const uint4 *src = reinterpret_cast<const uint4 *>(words_sec);
    uint4 *dst = reinterpret_cast<uint4 *>(out);
    const uint32_t nv = (n + 15) >> 4;
    uint32_t i = lane;
    for (; i + 96 < nv; i += 128) {                                    // four loads in flight per lane
        const uint4 a = src[i], b = src[i + 32], c = src[i + 64], d = src[i + 96];
        dst[i] = a; dst[i + 32] = b; dst[i + 64] = c; dst[i + 96] = d;
    }
    for (; i < nv; i += 32) dst[i] = src[i];
    if ((n & 1u) && lane == 0 && words_sec[n] != 0) ok = false;
    return __all_sync(0xFFFFFFFFu, ok);
}

// A CONST stream (FORMAT.md section 2, mode 2): n copies of the symbol in the low byte of the stream's one word.
// The stream areas of a slot are 16-byte aligned and padded, so the warp stores whole uint4s. The unused rANS states
// must be 2^16 and the word's high byte 0.
__device__ inline bool fill_const_stream(uint32_t x, uint32_t n, const uint8_t *words_sec, uint8_t *out, uint32_t lane)
{
    const uint32_t w = *reinterpret_cast<const uint16_t *>(words_sec);
    const bool ok = x == kRansL && (w >> 8) == 0;
    const uint32_t v = (w & 0xFFu) * 0x01010101u;
    uint4 *dst = reinterpret_cast<uint4 *>(out);
    for (uint32_t i = lane; i < (n + 15) >> 4; i += 32) dst[i] = make_uint4(v, v, v, v);
    return __all_sync(0xFFFFFFFFu, ok);
}

// One (block, stream) unit, by one warp: stream s of block blk into slot bi. Output: the slot's stream
// area and bad flag; with write_hdr also the record header fields in the slot header.
__device__ inline void decode_unit(const Container &cv, const SlotLayout &sl, uint8_t *slots, uint64_t blk, uint32_t bi,
                                   int s, bool write_hdr, const WarpSmem &ws, uint32_t lane, Control *ctl)
{
    uint8_t *slot = slots + (size_t)bi * sl.stride;
    SlotHdr *hdr = reinterpret_cast<SlotHdr *>(slot + sl.o_hdr);
    const Record r = open_record(cv, blk);
    bool ok = r.ok;
    // (stored by every lane - same address, same value, one transaction - rather than under a leader branch)
    if (write_hdr && ok) {
        hdr->n_seq = r.n_seq; hdr->n_lit = r.n_lit; hdr->block_len = r.block_len;
        hdr->n_extras = r.n_extras; hdr->off_nbytes = r.off_nbytes;
        hdr->extras_off = r.extras_off; hdr->tags_off = r.tags_off;
        const uint64_t ro = (uint64_t)(r.rec - cv.payload);
        hdr->rec_lo = (uint32_t)ro; hdr->rec_hi = (uint32_t)(ro >> 32);
    }
    if (ok) {
        // a stream longer than its slot area cannot occur once open() has found max_n_seq,
        // but the check keeps the store loop in bounds for any input
        const uint32_t cap = s == LIT ? kB : (s == LEN ? 2 * sl.ms : cv.W * sl.ms);
        const uint32_t ns = s == LIT ? r.n_sym[LIT] : (s == LEN ? r.n_sym[LEN] : r.n_sym[OFF]);
        if (ns > cap) ok = false;
    }
    if (ok) {
        uint8_t *out = slot + (s == LIT ? sl.o_lit : (s == LEN ? sl.o_len : sl.o_off));
        const uint32_t n = s == LIT ? r.n_sym[LIT] : (s == LEN ? r.n_sym[LEN] : r.n_sym[OFF]);
        const uint32_t nw = s == LIT ? r.n_words[LIT] : (s == LEN ? r.n_words[LEN] : r.n_words[OFF]);
        const uint32_t to = s == LIT ? r.tbl_off[LIT] : (s == LEN ? r.tbl_off[LEN] : r.tbl_off[OFF]);
        const uint32_t tb = s == LIT ? r.tbl_bytes[LIT] : (s == LEN ? r.tbl_bytes[LEN] : r.tbl_bytes[OFF]);
        const uint32_t wo = s == LIT ? r.words_off[LIT] : (s == LEN ? r.words_off[LEN] : r.words_off[OFF]);
        const uint32_t x0 = cv.states[(blk * 3 + (uint64_t)s) * kLanes + lane];
        const uint32_t is_raw = s == LIT ? r.raw[LIT] : (s == LEN ? r.raw[LEN] : r.raw[OFF]);
        if (is_raw == 1u) ok = copy_raw_stream(x0, n, r.rec + wo, out, lane);
        else if (is_raw == 2u) ok = fill_const_stream(x0, n, r.rec + wo, out, lane);
        else ok = decode_stream(x0, n, nw, r.rec + to, tb, r.rec + wo, out, ws, lane);
        if (!ok && leader()) raise(ctl, kStEntropy, blk);
    } else if (leader()) {
        raise(ctl, kStRecord, blk);
    }
    hdr->bad[s] = ok ? 0u : 1u;
    __syncwarp();
}

// Kernel: every warp takes (block, stream) units from a counter until none is left.
//   list != nullptr: the blocks are list[0 .. min(*n_list, max_slots)) (isolated path);
//   else:            the blocks are first .. first+count-1.
// Unit u -> stream u / nb in the order LIT, OFF, LEN; block index u % nb (= slot). Output: the slot's areas.
__global__ void __launch_bounds__(32 * kEntropyWarps) k_entropy(Container cv, SlotLayout sl, uint8_t *slots, const uint64_t *list,
                                                 const uint32_t *n_list, uint32_t max_slots, uint64_t first,
                                                 uint32_t count, Control *ctl, uint32_t reset_watermark, unsigned long long wm_init)
{
    extern __shared__ __align__(1024) uint8_t smem_entropy[];
    const uint32_t lane = lane_id(), warp = threadIdx.x >> 5;
    // decode_all / decode_range: the first launch of a call re-arms the watermark (0, resp. the first block of the range)
    if (reset_watermark && blockIdx.x == 0 && threadIdx.x == 0) ctl->watermark = wm_init;
    WarpSmem ws;
    {
        const uint32_t a0 = (uint32_t)__cvta_generic_to_shared(smem_entropy);
        const uint32_t pad = (0u - a0) & (kT8Bytes - 1);              // t8 region 4096-aligned in the shared window
        uint8_t *base = smem_entropy + pad;
        ws.t8 = base + warp * kT8Bytes;
        ws.syml = reinterpret_cast<uint2 *>(base + kEntropyWarps * kT8Bytes + warp * kSymlBytes);
        ws.ring = base + kEntropyWarps * (kT8Bytes + kSymlBytes) + warp * kRingBytes;
        ws.a_t8 = (uint32_t)__cvta_generic_to_shared(ws.t8);
        ws.a_syml = (uint32_t)__cvta_generic_to_shared(ws.syml);
        ws.a_ring = (uint32_t)__cvta_generic_to_shared(ws.ring);
    }
    uint32_t nb = count;
    if (list) { nb = *n_list; if (nb > max_slots) nb = max_slots; }
    const uint32_t n_units = 3 * nb;
    for (;;) {
        uint32_t u = 0;
        if (leader()) u = atomicAdd(&ctl->unit, 1u);
        u = __shfl_sync(0xFFFFFFFFu, u, 0);
        if (u >= n_units) break;
        // longest first: all LIT streams, then OFF, then LEN (balances the tail of the launch)
        const uint32_t so = u / nb, bi = u - so * nb;
        const int s = so == 0 ? LIT : (so == 1 ? OFF : LEN);
        decode_unit(cv, sl, slots, list ? list[bi] : first + bi, bi, s, s == LIT, ws, lane, ctl);
    }
    // last warp out re-arms the counters for the next launch
    if (lane == 0) {
        const uint32_t total = gridDim.x * (blockDim.x >> 5);
        __threadfence();
        if (atomicAdd(&ctl->unit_exit, 1u) == total - 1) {
            ctl->unit = 0;
            ctl->unit_exit = 0;
            __threadfence();
        }
    }
}

// Open-time scan: validate every block record header and find the largest n_seq.
__global__ void k_scan_records(Container cv, Control *ctl)
{
    const uint64_t b = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= cv.n_blocks) return;
    const Record r = open_record(cv, b);
    if (!r.ok) { raise(ctl, kStRecord, b); return; }
    atomicMax(&ctl->max_n_seq, r.n_seq);
}

// Test hook: copy decoded streams out of the slots into the caller's fixed-stride arrays.
__global__ void k_export_streams(Container cv, SlotLayout sl, const uint8_t *slots, uint64_t first, uint32_t count,
                                 uint8_t *d_lit, uint8_t *d_len, uint8_t *d_off)
{
    const uint32_t bi = blockIdx.x;
    if (bi >= count) return;
    const Record r = open_record(cv, first + bi);
    if (!r.ok) return;
    const uint8_t *slot = slots + (size_t)bi * sl.stride;
    for (uint32_t i = threadIdx.x; i < r.n_sym[LIT]; i += blockDim.x) d_lit[(size_t)bi * kB + i] = slot[sl.o_lit + i];
    for (uint32_t i = threadIdx.x; i < r.n_sym[LEN]; i += blockDim.x) d_len[(size_t)bi * (kB / 2) + i] = slot[sl.o_len + i];
    for (uint32_t i = threadIdx.x; i < r.n_sym[OFF]; i += blockDim.x) d_off[(size_t)bi * (2 * kB) + i] = slot[sl.o_off + i];
}

}  // namespace aceapex
