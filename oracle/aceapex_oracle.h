/*
 * ORACLE — TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, obviously-correct CPU implementation of the ACEAPEX-style two-layer codec of
 * arxiv/paper_2606_24531 in the container format of /FORMAT.md: an encoder (greedy hash-chain
 * global match search, absolute offsets, min match 4; BASELINE.json north_star) and two
 * independent decoders. Only tests/, __graft_entry__.smoke() and bench.py (its input preparation
 * and its cpu_baseline / --impl reference legs) may use anything under oracle/. It shares no
 * code with paper_2606_24531_b200/ (the CUDA path): every format constant is restated here from
 * FORMAT.md.
 *
 * Pins (tests/, -m "not gpu"): hand-computed rANS states/words, brute-force
 * round trips on tiny alphabets, the information identity, round-trip identity on all profiles
 * and adversarial sizes, decoder #1 == decoder #2 on every block, the closed form for N equal
 * bytes, the validator's src+len<=dst / tag / depth / window invariants, FNV-1a-64 standard
 * vectors. Parity unpinned: the paper's printed hashes and timings need its
 * dataset and code, which are absent.
 */
#ifndef ACEAPEX_ORACLE_H
#define ACEAPEX_ORACLE_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

enum {
    ORA_OK = 0,
    ORA_E_ARG = -1,      /* bad argument */
    ORA_E_FORMAT = -2,   /* bad magic / version / header field */
    ORA_E_CAPACITY = -3, /* output buffer too small */
    ORA_E_CORRUPT = -4,  /* container violates a validity rule of FORMAT.md */
    ORA_E_RANGE = -5,    /* block id / coordinate out of range */
    ORA_E_NOMEM = -6,
    ORA_E_PROMISE = -7   /* valid stream, but a header promise (D, R, tags) does not hold */
};

enum { ORA_LIT = 0, ORA_LEN = 1, ORA_OFF = 2 };

/* ---- entropy layer (FORMAT.md section 3; PAPER.md:33, :124 ref [6]) ---- */

/* FORMAT.md section 3 "Quantiser". count[256] -> freq[256], sum 4096 (all zero if n == 0). */
void ora_quantise(const uint32_t count[256], uint16_t freq[256]);

/* Interleaved rANS over `lanes` (1..32) states. words_out needs n entries at most.
 * states_out[lanes] receives the final encoder states. Returns ORA_OK or ORA_E_ARG
 * (a symbol with freq 0, or sum != 4096). */
int ora_rans_encode(const uint8_t *sym, size_t n, const uint16_t freq[256], uint32_t lanes,
                    uint32_t *states_out, uint16_t *words_out, size_t *n_words_out);

/* Sequential-semantics decoder of FORMAT.md section 3. Checks w == n_words and all states == 65536
 * at the end (ORA_E_CORRUPT otherwise). */
int ora_rans_decode(const uint32_t *states, uint32_t lanes, const uint16_t *words, size_t n_words,
                    const uint16_t freq[256], uint8_t *sym_out, size_t n);

/* FNV-1a 64-bit ("FNV hash"; reading A6). */
uint64_t ora_fnv1a64(const void *data, size_t n);

/* ---- encoder (north_star: greedy hash-chain, min match 4, absolute offsets) ---- */

typedef struct {
    uint32_t min_match;    /* accept threshold T >= 4 (format minimum is 4) */
    uint32_t chain_depth;  /* candidates tried per chain, newest first (default 32) */
    uint32_t max_depth;    /* D: bound on copy-hop depth of every byte; 0 = unbounded */
    uint32_t window;       /* R: see FORMAT.md header; 0 = none */
    uint32_t max_level;    /* cap on the in-block tag, 1..15 (default 15) */
    uint32_t offset_width; /* 4 or 8 */
    uint32_t threads;      /* worker threads for the parse (result does not depend on it) */
    uint32_t batch;        /* blocks parsed against one snapshot of the global table when R > 0
                              (default 64; part of the encoder's definition, not of the format) */
    uint32_t raw_slack_pct; /* selective entropy (FORMAT.md section 2 "modes"): a stream is stored
                              RAW when n_sym * 100 <= (tbl_bytes + 2 * n_words) * (100 + raw_slack_pct), i.e.
                              when rANS saves less than that margin. Default 0: RAW only where rANS does not
                              shrink the stream. 0xFFFFFFFF: never RAW. */
    uint32_t max_fanout;   /* F: the matches of a block read from at most F distinct earlier blocks (seek-aware
                              policy; header promise, FORMAT.md section 1); 0 = unbounded */
    uint32_t long_hash;    /* 0, or 9..16: bytes keyed by a second global hash table that is probed first
                              (SURVEY.md reading A14: 12) */
    uint32_t long_chain;   /* candidates tried on the long-hash chain (default 16) */
    uint32_t max_seq;      /* at most this many sequences per block, the rest of a block is literals; 0 = the format
                              limit (4096) */
} ora_enc_params;

typedef struct {
    uint64_t n_seq, n_lit, match_bytes, intra_match_bytes, n_extras;
    uint64_t n_sym[3], n_words[3], table_bytes;
    uint32_t max_depth_seen, max_level_seen;
    uint64_t n_raw[3];     /* streams stored RAW, per stream id */
    uint64_t n_const[3];   /* streams stored CONST, per stream id */
} ora_enc_stats;

/* the block_log2 this library was compiled for (14 unless built with -DORA_BLOG) */
int ora_block_log2(void);

void ora_enc_params_default(ora_enc_params *p);
size_t ora_encode_bound(size_t n);
int ora_encode(const uint8_t *in, size_t n, const ora_enc_params *p, uint8_t *out, size_t cap,
               size_t *out_len, ora_enc_stats *stats /* may be NULL */);

/* ---- container access ---- */

typedef struct {
    uint64_t total_len, n_blocks, payload_off, container_bytes;
    uint32_t offset_width, max_depth, window, max_level, min_match_policy, max_fanout;
} ora_info;

int ora_info_get(const uint8_t *c, size_t clen, ora_info *out);

/* Entropy-decode one block's three streams (decoder #1 steps 2.1-2.2). Each out buffer may be
 * NULL; capacities: lit 16384, len 8192, off 32768 bytes, extras 8192 u16, tags 4096 bytes
 * (one tag per byte, unpacked). */
typedef struct {
    uint32_t n_seq, n_lit, n_extras, off_nbytes;
    uint32_t n_sym[3], n_words[3];
} ora_block_hdr;
int ora_decode_streams(const uint8_t *c, size_t clen, uint64_t block, ora_block_hdr *hdr,
                       uint8_t *lit, uint8_t *len, uint8_t *off, uint16_t *extras, uint8_t *tags);

/* Parsed tokens of a block (decoder #1 step 2.3): per sequence lit_len, match_len, src.
 * Arrays need 4096 entries. */
int ora_decode_tokens(const uint8_t *c, size_t clen, uint64_t block, uint32_t *n_seq,
                      uint32_t *lit_len, uint32_t *match_len, uint64_t *src, uint8_t *tags);

/* Decoder #1: sequential, block order (defines decode_all). Writes out[0,total_len). */
int ora_decode_all(const uint8_t *c, size_t clen, uint8_t *out, size_t cap);

/* The same decoder with the entropy stage (steps 2.1-2.3, independent per block) spread over
 * `threads` host threads and the match stage (step 2.4) in block order on one thread; the multi-core CPU
 * baseline of SURVEY.md section 8(d). Bit-identical to ora_decode_all. */
int ora_decode_all_mt(const uint8_t *c, size_t clen, uint8_t *out, size_t cap, uint32_t threads);

/* Decoder #2: per-byte origin chase (defines seek / decode_blocks). Independent algorithm.
 * Writes only dst[0, block_len). The context memoises parsed blocks. */
typedef struct ora_iso ora_iso;
int ora_iso_open(const uint8_t *c, size_t clen, ora_iso **out);
int ora_iso_decode(ora_iso *ctx, uint64_t block, uint8_t *dst, size_t cap, uint32_t *block_len,
                   uint32_t *max_hops /* may be NULL: longest chase in this block */);
void ora_iso_close(ora_iso *ctx);

/* Validator: every rule of FORMAT.md section 4 "Validity", recomputing tags, byte depths and the
 * window rule. Returns ORA_OK, ORA_E_CORRUPT (invalid stream) or ORA_E_PROMISE. */
typedef struct {
    uint64_t n_seq, n_matches_cross, n_matches_intra, n_matches_spanning;
    uint32_t max_depth_seen, max_level_seen, min_match_seen, max_src_blocks_per_block;
    double mean_src_blocks_per_block;
} ora_validate_report;
int ora_validate(const uint8_t *c, size_t clen, ora_validate_report *rep /* may be NULL */);

const char *ora_strerror(int code);

#ifdef __cplusplus
}
#endif
#endif
