// FORMAT.md restated for the CUDA path (container, index, block record). Shares nothing with
// oracle/: every constant below is written out from FORMAT.md sections 1-2.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace aceapex {

// FORMAT.md section 1: block_log2. 14 = 16384 bytes per block; -DACEAPEX_BLOCK_LOG2=12..15 builds the
// library for another block size (block-size sweep; `bench.py --sweep`). 16 would not fit the
// record header's 16-bit n_lit, nor the 16-bit positions the kernels pack in pairs.
#ifndef ACEAPEX_BLOCK_LOG2
#define ACEAPEX_BLOCK_LOG2 14
#endif
constexpr uint32_t kBlockLog2 = ACEAPEX_BLOCK_LOG2;
static_assert(kBlockLog2 >= 12 && kBlockLog2 <= 15, "block size 4 .. 32 KiB");
constexpr uint32_t kB = 1u << kBlockLog2;
constexpr uint32_t kMaxSeq = kB / 4;           // n_seq <= block size / 4: a sequence is at least 4 bytes (FORMAT.md section 2)
constexpr uint32_t kLanes = 32;                // rANS lanes per stream
constexpr uint32_t kProbBits = 12;             // 12-bit quantised frequencies
constexpr uint32_t kM = 1u << kProbBits;       // 4096
constexpr uint32_t kRansL = 1u << 16;          // state interval [2^16, 2^32)
constexpr uint32_t kHeaderBytes = 64;
constexpr uint32_t kRecHeaderBytes = 32;
enum Stream : int { LIT = 0, LEN = 1, OFF = 2 };

// sticky device status bits (Control::status)
constexpr uint32_t kStRecord = 1u;   // block record header / section layout invalid
constexpr uint32_t kStEntropy = 2u;  // table sum != 4096, word count or final state mismatch
constexpr uint32_t kStTokens = 4u;   // token sums, escapes, src+len<=dst violated
constexpr uint32_t kStChase = 8u;    // isolated decode: chase left the valid range / depth promise broken

struct Container {
    const uint8_t *base;       // DEVICE, 16-byte aligned
    const uint64_t *rec_off;   // n_blocks+1 entries, relative to payload
    const uint32_t *states;    // [n_blocks][3][32]
    const uint8_t *payload;
    uint64_t total_len, n_blocks, payload_bytes;
    uint32_t W, D, R, max_level;
};

// One block record located section by section (FORMAT.md section 2).
struct Record {
    const uint8_t *rec;
    uint32_t block_len, n_seq, n_lit, n_extras, off_nbytes;
    uint32_t n_sym[3], n_words[3], tbl_bytes[3];
    uint32_t raw[3];           // stream mode (FORMAT.md section 2; PAPER.md:94 selective entropy): 0 rANS, 1 RAW, 2 CONST
    uint32_t tbl_off[3], extras_off, tags_off, words_off[3];
    bool ok;
};

__host__ __device__ inline uint32_t pad16(uint32_t x) { return (x + 15u) & ~15u; }

__device__ inline uint32_t block_len_of(const Container &cv, uint64_t b)
{
    uint64_t start = b << kBlockLog2;
    uint64_t rest = cv.total_len - start;
    return rest < kB ? (uint32_t)rest : kB;
}

// Parse and validate the 32-byte record header of block b (FORMAT.md section 2).
__device__ inline Record open_record(const Container &cv, uint64_t b)
{
    Record r;
    r.ok = false;
    r.rec = nullptr;
    r.block_len = block_len_of(cv, b);
    r.n_seq = r.n_lit = r.n_extras = r.off_nbytes = 0;
    for (int s = 0; s < 3; s++) { r.n_sym[s] = r.n_words[s] = r.tbl_bytes[s] = r.tbl_off[s] = r.words_off[s] = r.raw[s] = 0; }
    r.extras_off = r.tags_off = 0;
    const uint64_t o0 = cv.rec_off[b], o1 = cv.rec_off[b + 1];
    if (o1 < o0 || (o0 & 15) || (o1 & 15) || o1 - o0 < kRecHeaderBytes || o1 > cv.payload_bytes) return r;
    if (o1 - o0 > (1u << 20)) return r;   // a record of a 16 KiB block is far below 1 MiB
    const uint32_t rec_bytes = (uint32_t)(o1 - o0);
    const uint8_t *rec = cv.payload + o0;
    r.rec = rec;
    const uint4 h0 = *reinterpret_cast<const uint4 *>(rec);
    const uint4 h1 = *reinterpret_cast<const uint4 *>(rec + 16);
    r.n_seq = h0.x & 0xFFFFu;
    r.n_lit = h0.x >> 16;
    r.n_extras = h0.y & 0xFFFFu;
    r.off_nbytes = (h0.y >> 16) & 0xFFu;
    const uint32_t modes = h0.y >> 24;
    r.n_words[LIT] = h0.z;
    r.n_words[LEN] = h0.w;
    r.n_words[OFF] = h1.x;
    r.tbl_bytes[LIT] = h1.y & 0xFFFFu;
    r.tbl_bytes[LEN] = h1.y >> 16;
    r.tbl_bytes[OFF] = h1.z & 0xFFFFu;
    if (r.n_seq > kMaxSeq || r.n_lit > r.block_len) return r;
    if (r.off_nbytes < 1 || r.off_nbytes > cv.W) return r;
    if (modes & 0xC0u) return r;                       // per stream: 0 = rANS, 1 = RAW, 2 = CONST; 3 and bits 6-7 reserved
    r.raw[LIT] = modes & 3u; r.raw[LEN] = (modes >> 2) & 3u; r.raw[OFF] = (modes >> 4) & 3u;
    if (r.raw[LIT] == 3u || r.raw[LEN] == 3u || r.raw[OFF] == 3u) return r;
    if (r.n_extras > 2 * r.n_seq) return r;
    r.n_sym[LIT] = r.n_lit;
    r.n_sym[LEN] = 2 * r.n_seq;
    r.n_sym[OFF] = r.off_nbytes * r.n_seq;
    uint32_t pos = kRecHeaderBytes;
    for (int s = 0; s < 3; s++) {
        pos = pad16(pos);
        r.tbl_off[s] = pos;
        if (r.tbl_bytes[s] > 32 + 512) return r;
        pos += r.tbl_bytes[s];
        if (r.raw[s] == 1u) {                          // RAW: no table; the symbols sit in the words section
            if (r.n_sym[s] == 0 || r.tbl_bytes[s] != 0 || r.n_words[s] != (r.n_sym[s] + 1) / 2) return r;
        } else if (r.raw[s] == 2u) {                   // CONST: no table; one word whose low byte is the symbol
            if (r.n_sym[s] == 0 || r.tbl_bytes[s] != 0 || r.n_words[s] != 1) return r;
        } else {
            if ((r.n_sym[s] == 0) != (r.tbl_bytes[s] == 0)) return r;
            if (r.n_words[s] > r.n_sym[s]) return r;
        }
    }
    pos = pad16(pos); r.extras_off = pos; pos += 2 * r.n_extras;
    pos = pad16(pos); r.tags_off = pos; pos += (r.n_seq + 1) / 2;
    for (int s = 0; s < 3; s++) {
        pos = pad16(pos);
        r.words_off[s] = pos;
        pos += 2 * r.n_words[s];
    }
    if (pad16(pos) != rec_bytes) return r;
    r.ok = true;
    return r;
}

// ---------------------------------------------------------------------------------------------
// Scratch layout (host computes, kernels consume).

struct Control {
    unsigned long long first_bad;   // lowest block id that raised a status bit (atomicMin)
    unsigned long long watermark;   // decode_all: number of leading blocks complete
    unsigned long long rsv0;
    uint32_t status;                // sticky kSt* bits
    uint32_t ticket, ticket_exit;   // decode_all match kernel: ordered block hand-out
    uint32_t unit, unit_exit;       // entropy kernel: (block, stream) unit hand-out
    uint32_t rsv1;
    uint32_t max_n_seq;             // open-time scan result
    // fused isolated decode (seek.cuh): counters, double-buffered by round / hop parity
    uint32_t rsv3[2];
    uint32_t round_n_list[2];       // distinct blocks claimed so far in the round (by round parity)
    uint32_t rsv2[3];
    unsigned long long hop_pending[2];   // bytes still chasing after the hop (by hop parity)
    uint32_t pad[8];
};
static_assert(sizeof(Control) == 128, "Control layout");

// A slot holds one block's decoded token streams and, for the isolated path, its parsed tokens.
struct SlotLayout {
    uint32_t ms;         // capacity in sequences (container max n_seq rounded up to 16)
    uint32_t o_hdr;      // SlotHdr
    uint32_t o_lit;      // u8  [16384]   decoded LIT stream
    uint32_t o_len;      // u8  [2*ms]    decoded LEN stream
    uint32_t o_off;      // u8  [W*ms]    decoded OFF stream
    uint32_t o_start;    // u16 [ms+16]   seq_start[k]: in-block output offset of sequence k's literal run
    uint32_t o_dst;      // u16 [ms]      dst[k]: in-block output offset of match k
    uint32_t o_litpos;   // u16 [ms+16]   index into LIT of sequence k's first literal
    uint32_t o_src;      // u64 [ms]      absolute source position of match k
    uint32_t stride;     // bytes per slot, multiple of 256
};

struct SlotHdr {
    uint32_t bad[3];     // per stream: entropy decode failed (bad[LIT] also: record header invalid)
    uint32_t n_seq, n_lit, block_len;
    uint32_t parsed_ok;  // isolated decode: tokens parsed and valid
    // record header fields, written by the entropy kernel's LIT unit so that the match kernel needs
    // one 64-byte load instead of the rec_off -> record header chain
    uint32_t n_extras, off_nbytes, extras_off, tags_off;
    uint32_t rec_lo, rec_hi;   // record offset relative to the payload
    uint32_t need_lit;         // isolated decode: some chased byte ends on a literal of this block
    uint32_t pad[2];
};
static_assert(sizeof(SlotHdr) == 64, "SlotHdr layout");

__host__ inline SlotLayout make_slot_layout(uint32_t max_n_seq, uint32_t W)
{
    SlotLayout L;
    uint32_t ms = (max_n_seq + 15u) & ~15u;
    if (ms < 16) ms = 16;
    L.ms = ms;
    uint32_t p = 0;
    L.o_hdr = p; p += 64;
    L.o_lit = p; p += kB;
    L.o_len = p; p += 2 * ms;
    L.o_off = p; p += W * ms;
    L.o_start = p; p += 2 * (ms + 16);
    L.o_dst = p; p += 2 * ms;
    L.o_litpos = p; p += 2 * (ms + 16);
    p = (p + 7u) & ~7u;
    L.o_src = p; p += 8 * ms;
    L.stride = (p + 255u) & ~255u;
    return L;
}

struct Scratch {
    Control *ctl;
    uint32_t *done;      // [n_blocks] epoch of the decode_all call that completed the block
    uint32_t *mark;      // [n_blocks] tag of the isolated-decode round that claimed the block
    unsigned long long *slot_of;   // [n_blocks] round tag << 32 | slot index assigned in that round
    uint64_t *list;      // [n_slots]  block id held by each slot in this round
    uint64_t *ids;       // [n_targets] target block ids of the current group
    uint8_t *slots;      // n_slots * stride
    uint64_t *pend;      // [n_targets][16384] absolute position still to be chased, literal request, or kDone
    uint64_t n_slots, n_targets;
};

constexpr unsigned long long kDone = ~0ull;

__device__ inline void raise(Control *ctl, uint32_t bit, uint64_t blk)
{
    atomicOr(&ctl->status, bit);
    atomicMin(&ctl->first_bad, (unsigned long long)blk);
}

}  // namespace aceapex
