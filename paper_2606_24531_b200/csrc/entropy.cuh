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

constexpr uint32_t kTblWords = kM;          // packed decode table: one u32 per slot
constexpr uint32_t kSymListWords = 256;     // present symbols, packed
constexpr uint32_t kEntropyWarpSmemWords = kTblWords + kSymListWords;

__device__ inline uint32_t lane_id() { return threadIdx.x & 31u; }

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

// Build the 4096-entry packed decode table of one stream in shared memory.
// entry = sym | (f-1) << 8 | (slot - c[sym]) << 20, so that x' = f*(x>>12) + (slot - c).
// Returns false (warp-uniform) if the table section is invalid (FORMAT.md section 3 "Table").
__device__ inline bool build_table(const uint8_t *tbl_sec, uint32_t tbl_bytes, uint32_t *tbl, uint32_t *syml,
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
    if (__any_sync(0xFFFFFFFFu, bad)) return false;      // also bounds every f before the scan
    uint32_t total;
    uint32_t c = warp_excl_scan(sum, lane, total);
    if (total != kM) return false;
    {
        uint32_t j = first;
#pragma unroll
        for (int k = 0; k < 8; k++)
            if (bm >> k & 1u) {
                syml[j++] = (8 * lane + k) | (f[k] - 1) << 8 | c << 20;   // c <= 4095
                c += f[k];
            }
    }
    __syncwarp();
    for (uint32_t j = 0; j < n_present; j++) {
        const uint32_t e = syml[j];
        const uint32_t fm1 = (e >> 8) & 0xFFFu, c0 = e >> 20, lo = e & 0xFFFFFu;
        for (uint32_t k = lane; k <= fm1; k += 32) tbl[c0 + k] = lo | k << 20;
    }
    __syncwarp();
    return true;
}

// Decode stream s of block `blk` into out[0, n_sym). One warp. Returns true (warp-uniform) on
// success; false if the table or the rANS end conditions are violated (then out is unspecified
// but never written beyond n_sym).
__device__ inline bool decode_stream(const Container &cv, const Record &r, int s, uint64_t blk, uint8_t *out,
                                     uint32_t *tbl, uint32_t *syml, uint32_t lane)
{
    const uint32_t n = r.n_sym[s], n_words = r.n_words[s];
    uint32_t x = cv.states[(blk * 3 + (uint64_t)s) * kLanes + lane];
    if (n == 0) return __all_sync(0xFFFFFFFFu, x == kRansL) && n_words == 0;
    if (!build_table(r.rec + r.tbl_off[s], r.tbl_bytes[s], tbl, syml, lane)) return false;
    const uint16_t *words = reinterpret_cast<const uint16_t *>(r.rec + r.words_off[s]);
    const uint32_t lt = (1u << lane) - 1u;
    uint32_t wpos = 0;
    bool overrun = false;
    const uint32_t rounds = (n + 31u) >> 5;
    for (uint32_t rd = 0; rd < rounds; rd++) {
        const uint32_t i = (rd << 5) + lane;
        const bool active = i < n;
        bool need = false;
        uint32_t sym = 0;
        if (active) {
            const uint32_t e = tbl[x & (kM - 1)];
            sym = e & 0xFFu;
            x = (((e >> 8) & 0xFFFu) + 1u) * (x >> kProbBits) + (e >> 20);
            need = x < kRansL;
        }
        const uint32_t mask = __ballot_sync(0xFFFFFFFFu, need);
        if (need) {
            const uint32_t idx = wpos + __popc(mask & lt);
            uint32_t w = 0;
            if (idx < n_words) w = __ldg(words + idx); else overrun = true;
            x = (x << 16) | w;
        }
        wpos += __popc(mask);
        if (active) out[i] = (uint8_t)sym;
    }
    const bool good = !overrun && x == kRansL;
    return __all_sync(0xFFFFFFFFu, good) && wpos == n_words;
}

// Kernel: every warp takes (block, stream) units from a counter until none is left.
//   list != nullptr: the blocks are list[0 .. min(*n_list, max_slots)) (isolated path);
//   else:            the blocks are first .. first+count-1.
// Unit u -> block index u/3 (= slot), stream u%3. Output: the slot's LIT/LEN/OFF areas.
__global__ void __launch_bounds__(128) k_entropy(Container cv, SlotLayout sl, uint8_t *slots, const uint64_t *list,
                                                 const uint32_t *n_list, uint32_t max_slots, uint64_t first,
                                                 uint32_t count, Control *ctl)
{
    extern __shared__ uint32_t smem_u32[];
    const uint32_t lane = lane_id(), warp = threadIdx.x >> 5;
    uint32_t *tbl = smem_u32 + warp * kEntropyWarpSmemWords;
    uint32_t *syml = tbl + kTblWords;
    uint32_t nb = count;
    if (list) { nb = *n_list; if (nb > max_slots) nb = max_slots; }
    const uint32_t n_units = 3 * nb;
    for (;;) {
        uint32_t u = 0;
        if (lane == 0) u = atomicAdd(&ctl->unit, 1u);
        u = __shfl_sync(0xFFFFFFFFu, u, 0);
        if (u >= n_units) break;
        const uint32_t bi = u / 3;
        const int s = (int)(u - 3 * bi);
        const uint64_t blk = list ? list[bi] : first + bi;
        uint8_t *slot = slots + (size_t)bi * sl.stride;
        SlotHdr *hdr = reinterpret_cast<SlotHdr *>(slot + sl.o_hdr);
        const Record r = open_record(cv, blk);
        bool ok = r.ok;
        if (ok) {
            // a stream longer than its slot area cannot occur once open() has found max_n_seq,
            // but the check keeps the store loop in bounds for any input
            const uint32_t cap = s == LIT ? kB : (s == LEN ? 2 * sl.ms : cv.W * sl.ms);
            if (r.n_sym[s] > cap) ok = false;
        }
        if (ok) {
            uint8_t *out = slot + (s == LIT ? sl.o_lit : (s == LEN ? sl.o_len : sl.o_off));
            ok = decode_stream(cv, r, s, blk, out, tbl, syml, lane);
            if (!ok && lane == 0) raise(ctl, kStEntropy, blk);
        } else if (lane == 0) {
            raise(ctl, kStRecord, blk);
        }
        if (lane == 0) hdr->bad[s] = ok ? 0u : 1u;
        __syncwarp();
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
    for (uint32_t i = threadIdx.x; i < r.n_sym[LEN]; i += blockDim.x) d_len[(size_t)bi * 8192 + i] = slot[sl.o_len + i];
    for (uint32_t i = threadIdx.x; i < r.n_sym[OFF]; i += blockDim.x) d_off[(size_t)bi * 32768 + i] = slot[sl.o_off + i];
}

}  // namespace aceapex
