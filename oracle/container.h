/* ORACLE (test infrastructure) — container and record parsing, FORMAT.md sections 1-2.
 * Internal to oracle/. */
#ifndef ACEAPEX_ORACLE_CONTAINER_H
#define ACEAPEX_ORACLE_CONTAINER_H

#include "aceapex_oracle.h"
#include <string.h>

/* FORMAT.md section 1: block_log2. 14 (16 KiB) unless the library is built with -DORA_BLOG=12..15 for the
 * block-size sweep ("block size ... governs how many independent parsers the format exposes").
 * 16 would need more than the record header's 16-bit n_lit field. */
#ifndef ORA_BLOG
#define ORA_BLOG 14
#endif
#if ORA_BLOG < 12 || ORA_BLOG > 15
#error "ORA_BLOG must be 12..15"
#endif
#define ORA_B (1u << ORA_BLOG)
#define ORA_MAX_SEQ (ORA_B / 4u)          /* a sequence is at least 4 bytes long */
#define ORA_HDR_BYTES 64u
#define ORA_REC_HDR_BYTES 32u

static inline uint16_t rd16(const uint8_t *p) { return (uint16_t)(p[0] | (p[1] << 8)); }
static inline uint32_t rd32(const uint8_t *p)
{ return (uint32_t)p[0] | ((uint32_t)p[1] << 8) | ((uint32_t)p[2] << 16) | ((uint32_t)p[3] << 24); }
static inline uint64_t rd64(const uint8_t *p) { return (uint64_t)rd32(p) | ((uint64_t)rd32(p + 4) << 32); }
static inline void wr16(uint8_t *p, uint32_t v) { p[0] = (uint8_t)v; p[1] = (uint8_t)(v >> 8); }
static inline void wr32(uint8_t *p, uint32_t v) { wr16(p, v & 0xFFFF); wr16(p + 2, v >> 16); }
static inline void wr64(uint8_t *p, uint64_t v) { wr32(p, (uint32_t)v); wr32(p + 4, (uint32_t)(v >> 32)); }
static inline size_t pad16(size_t x) { return (x + 15) & ~(size_t)15; }

typedef struct {
    const uint8_t *c;
    size_t clen;
    ora_info info;
    const uint8_t *rec_off;  /* u64[n_blocks+1] */
    const uint8_t *states;   /* u32[n_blocks][3][32] */
} ora_container;

/* One block record, located section by section (FORMAT.md section 2). */
typedef struct {
    uint32_t block_len;
    uint32_t n_seq, n_lit, n_extras, off_nbytes, modes;
    uint32_t n_sym[3], n_words[3], tbl_bytes[3];
    const uint8_t *table[3], *extras, *tags, *words[3];
    uint32_t states[3][32];
} ora_record;

int ora_container_open(const uint8_t *c, size_t clen, ora_container *out);
int ora_record_open(const ora_container *k, uint64_t block, ora_record *r);
/* freq[256] from a table section; ORA_E_CORRUPT if the sum is not 4096 or sizes disagree */
int ora_table_read(const uint8_t *tbl, uint32_t tbl_bytes, uint16_t freq[256]);

/* tokens of one block after entropy decode + parse (decoder steps 2.1-2.3) */
typedef struct {
    uint32_t n_seq, n_lit, block_len, trailing;
    uint32_t lit_len[ORA_MAX_SEQ], match_len[ORA_MAX_SEQ];
    uint64_t src[ORA_MAX_SEQ];
    uint8_t tag[ORA_MAX_SEQ];
    uint8_t lit[ORA_B];
} ora_tokens;
int ora_tokens_decode(const ora_container *k, uint64_t block, ora_tokens *t);

#endif
