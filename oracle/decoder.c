/* ORACLE (test infrastructure) — the two decoders and the validator.
 *
 * Decoder #1 (ora_decode_all): sequential, block order; defines decode_all. Follows PAPER.md:27
 *   (literals + copies from absolute positions), :33 (per-block entropy entry), :76.
 * Decoder #2 (ora_iso_decode): per-byte origin chase; defines seek / decode_blocks. Follows
 *   PAPER.md:35 ("a match referencing absolute position p can be resolved as soon as the block
 *   containing p is available") and :45-51 (only the target block is written). DESIGN.md
 *   reading A7: the paper does not say how a seeked block obtains its source bytes; this decoder
 *   re-derives each byte from the compressed data of the block that owns it.
 * The two decoders share only the entropy decode + token parse of one block (ora_tokens_decode);
 * the match-layer logic is separate, and their agreement on every block is itself a pin.
 */
#include "container.h"

#include <stdlib.h>

/* ---------------------------------------------------------------- container / record parsing */

int ora_container_open(const uint8_t *c, size_t clen, ora_container *out)
{
    static const char magic[8] = { 'A', 'C', 'E', 'A', 'P', 'E', 'X', '1' };
    if (!c || !out) return ORA_E_ARG;
    if (clen < ORA_HDR_BYTES) return ORA_E_FORMAT;
    if (memcmp(c, magic, 8) != 0) return ORA_E_FORMAT;
    if (rd32(c + 8) != 1) return ORA_E_FORMAT;
    if (c[12] != ORA_BLOG || (c[13] != 4 && c[13] != 8) || c[14] != 32 || c[15] != 12) return ORA_E_FORMAT;
    ora_info *I = &out->info;
    I->offset_width = c[13];
    I->total_len = rd64(c + 16);
    I->n_blocks = rd64(c + 24);
    I->max_depth = rd32(c + 32);
    I->window = rd32(c + 36);
    I->max_level = rd32(c + 40);
    I->min_match_policy = rd32(c + 44) & 0xFFFFu;
    I->max_fanout = rd32(c + 44) >> 16;
    uint64_t index_off = rd64(c + 48);
    I->payload_off = rd64(c + 56);
    if (I->n_blocks != (I->total_len + ORA_B - 1) / ORA_B) return ORA_E_FORMAT;
    if (index_off != ORA_HDR_BYTES || I->max_level > 15) return ORA_E_FORMAT;
    if (I->n_blocks > ((uint64_t)1 << 40)) return ORA_E_FORMAT;
    uint64_t index_bytes = (I->n_blocks + 1) * 8 + I->n_blocks * 3 * 32 * 4;
    if (I->payload_off != pad16(ORA_HDR_BYTES + index_bytes) || I->payload_off > clen) return ORA_E_FORMAT;
    out->c = c;
    out->clen = clen;
    out->rec_off = c + ORA_HDR_BYTES;
    out->states = out->rec_off + (I->n_blocks + 1) * 8;
    I->container_bytes = I->payload_off + rd64(out->rec_off + I->n_blocks * 8);
    if (I->container_bytes > clen) return ORA_E_FORMAT;
    if (rd64(out->rec_off) != 0) return ORA_E_FORMAT;
    return ORA_OK;
}

int ora_info_get(const uint8_t *c, size_t clen, ora_info *out)
{
    ora_container k;
    int rc = ora_container_open(c, clen, &k);
    if (rc == ORA_OK) *out = k.info;
    return rc;
}

int ora_record_open(const ora_container *k, uint64_t block, ora_record *r)
{
    if (block >= k->info.n_blocks) return ORA_E_RANGE;
    uint64_t o0 = rd64(k->rec_off + block * 8), o1 = rd64(k->rec_off + (block + 1) * 8);
    if (o1 < o0 || (o0 & 15) || (o1 & 15) || o1 - o0 < ORA_REC_HDR_BYTES) return ORA_E_CORRUPT;
    if (k->info.payload_off + o1 > k->clen) return ORA_E_CORRUPT;
    const uint8_t *rec = k->c + k->info.payload_off + o0;
    size_t rec_bytes = (size_t)(o1 - o0);
    uint64_t start = block * ORA_B;
    r->block_len = (uint32_t)((k->info.total_len - start < ORA_B) ? (k->info.total_len - start) : ORA_B);
    r->n_seq = rd16(rec + 0);
    r->n_lit = rd16(rec + 2);
    r->n_extras = rd16(rec + 4);
    r->off_nbytes = rec[6];
    r->modes = rec[7];
    for (int s = 0; s < 3; s++) {
        r->n_words[s] = rd32(rec + 8 + 4 * s);
        r->tbl_bytes[s] = rd16(rec + 20 + 2 * s);
    }
    if (r->n_seq > ORA_MAX_SEQ || r->n_lit > r->block_len) return ORA_E_CORRUPT;
    if (r->off_nbytes < 1 || r->off_nbytes > k->info.offset_width) return ORA_E_CORRUPT;
    /* per stream 2 bits: 0 = rANS, 1 = RAW, 2 = CONST; 3 and bits 6-7 reserved */
    if (r->modes & 0xC0u) return ORA_E_CORRUPT;
    for (int s = 0; s < 3; s++) if (((r->modes >> (2 * s)) & 3u) == 3u) return ORA_E_CORRUPT;
    if (r->n_extras > 2 * r->n_seq) return ORA_E_CORRUPT;
    r->n_sym[ORA_LIT] = r->n_lit;
    r->n_sym[ORA_LEN] = 2 * r->n_seq;
    r->n_sym[ORA_OFF] = r->off_nbytes * r->n_seq;
    size_t pos = ORA_REC_HDR_BYTES;
    for (int s = 0; s < 3; s++) {
        pos = pad16(pos);
        r->table[s] = rec + pos;
        pos += r->tbl_bytes[s];
        const uint32_t mode = (r->modes >> (2 * s)) & 3u;
        if (mode == 1u) {                       /* RAW: no table, the symbols sit in the words section */
            if (r->n_sym[s] == 0 || r->tbl_bytes[s] != 0 || r->n_words[s] != (r->n_sym[s] + 1) / 2) return ORA_E_CORRUPT;
        } else if (mode == 2u) {                /* CONST: no table, one word whose low byte is the symbol */
            if (r->n_sym[s] == 0 || r->tbl_bytes[s] != 0 || r->n_words[s] != 1) return ORA_E_CORRUPT;
        } else {
            if ((r->n_sym[s] == 0) != (r->tbl_bytes[s] == 0)) return ORA_E_CORRUPT;
            if (r->n_words[s] > r->n_sym[s]) return ORA_E_CORRUPT;
        }
    }
    pos = pad16(pos); r->extras = rec + pos; pos += 2 * (size_t)r->n_extras;
    pos = pad16(pos); r->tags = rec + pos; pos += (r->n_seq + 1) / 2;
    for (int s = 0; s < 3; s++) {
        pos = pad16(pos);
        r->words[s] = rec + pos;
        pos += 2 * (size_t)r->n_words[s];
    }
    if (pad16(pos) != rec_bytes) return ORA_E_CORRUPT;
    for (int s = 0; s < 3; s++)
        for (int l = 0; l < 32; l++)
            r->states[s][l] = rd32(k->states + ((block * 3 + (uint64_t)s) * 32 + (uint64_t)l) * 4);
    return ORA_OK;
}

int ora_table_read(const uint8_t *tbl, uint32_t tbl_bytes, uint16_t freq[256])
{
    uint32_t n_present = 0, sum = 0, j = 0;
    memset(freq, 0, 256 * sizeof(uint16_t));
    if (tbl_bytes < 32) return ORA_E_CORRUPT;
    for (int s = 0; s < 256; s++) n_present += (tbl[s >> 3] >> (s & 7)) & 1u;
    if (tbl_bytes != 32 + 2 * n_present || n_present == 0) return ORA_E_CORRUPT;
    for (int s = 0; s < 256; s++) {
        if (!((tbl[s >> 3] >> (s & 7)) & 1u)) continue;
        uint32_t f = rd16(tbl + 32 + 2 * j++);
        if (f < 1 || f > 4096) return ORA_E_CORRUPT;
        freq[s] = (uint16_t)f;
        sum += f;
    }
    return sum == 4096 ? ORA_OK : ORA_E_CORRUPT;
}

/* decoder steps 2.1-2.2: entropy-decode one stream of a record */
static int stream_decode(const ora_record *r, int s, uint8_t *out)
{
    uint16_t freq[256];
    if (((r->modes >> (2 * s)) & 3u) == 2u) {   /* CONST (FORMAT.md section 2): n_sym copies of one symbol */
        for (int l = 0; l < 32; l++) if (r->states[s][l] != 65536u) return ORA_E_CORRUPT;
        if (r->words[s][1] != 0) return ORA_E_CORRUPT;                                    /* high byte of the word */
        memset(out, r->words[s][0], r->n_sym[s]);
        return ORA_OK;
    }
    if (((r->modes >> (2 * s)) & 3u) == 1u) {   /* RAW (FORMAT.md section 2): copy; states unused, must be 2^16 */
        for (int l = 0; l < 32; l++) if (r->states[s][l] != 65536u) return ORA_E_CORRUPT;
        memcpy(out, r->words[s], r->n_sym[s]);
        if ((r->n_sym[s] & 1u) && r->words[s][r->n_sym[s]] != 0) return ORA_E_CORRUPT;   /* pad byte of the last word */
        return ORA_OK;
    }
    if (r->n_sym[s] == 0) {
        for (int l = 0; l < 32; l++) if (r->states[s][l] != 65536u) return ORA_E_CORRUPT;
        return r->n_words[s] == 0 ? ORA_OK : ORA_E_CORRUPT;
    }
    int rc = ora_table_read(r->table[s], r->tbl_bytes[s], freq);
    if (rc != ORA_OK) return rc;
    /* words are 2-byte aligned inside a 16-byte aligned section; copy to be alignment-agnostic */
    uint16_t *w = (uint16_t *)malloc(sizeof(uint16_t) * (r->n_words[s] ? r->n_words[s] : 1));
    if (!w) return ORA_E_NOMEM;
    for (uint32_t i = 0; i < r->n_words[s]; i++) w[i] = rd16(r->words[s] + 2 * (size_t)i);
    rc = ora_rans_decode(r->states[s], 32, w, r->n_words[s], freq, out, r->n_sym[s]);
    free(w);
    return rc;
}

int ora_decode_streams(const uint8_t *c, size_t clen, uint64_t block, ora_block_hdr *hdr,
                       uint8_t *lit, uint8_t *len, uint8_t *off, uint16_t *extras, uint8_t *tags)
{
    ora_container k;
    ora_record r;
    int rc = ora_container_open(c, clen, &k);
    if (rc != ORA_OK) return rc;
    if ((rc = ora_record_open(&k, block, &r)) != ORA_OK) return rc;
    if (hdr) {
        hdr->n_seq = r.n_seq; hdr->n_lit = r.n_lit; hdr->n_extras = r.n_extras;
        hdr->off_nbytes = r.off_nbytes;
        for (int s = 0; s < 3; s++) { hdr->n_sym[s] = r.n_sym[s]; hdr->n_words[s] = r.n_words[s]; }
    }
    uint8_t *outs[3] = { lit, len, off };
    for (int s = 0; s < 3; s++)
        if (outs[s] && (rc = stream_decode(&r, s, outs[s])) != ORA_OK) return rc;
    if (extras) for (uint32_t i = 0; i < r.n_extras; i++) extras[i] = rd16(r.extras + 2 * (size_t)i);
    if (tags) for (uint32_t k2 = 0; k2 < r.n_seq; k2++) tags[k2] = (r.tags[k2 >> 1] >> ((k2 & 1) * 4)) & 15u;
    return ORA_OK;
}

/* decoder steps 2.1-2.3: entropy decode, then parse tokens (FORMAT.md section 4) */
int ora_tokens_decode(const ora_container *k, uint64_t block, ora_tokens *t)
{
    ora_record r;
    uint8_t len[2 * ORA_MAX_SEQ];
    uint8_t *off = NULL;
    int rc = ora_record_open(k, block, &r);
    if (rc != ORA_OK) return rc;
    t->n_seq = r.n_seq; t->n_lit = r.n_lit; t->block_len = r.block_len;
    if ((rc = stream_decode(&r, ORA_LIT, t->lit)) != ORA_OK) return rc;
    if ((rc = stream_decode(&r, ORA_LEN, len)) != ORA_OK) return rc;
    off = (uint8_t *)malloc(r.n_sym[ORA_OFF] ? r.n_sym[ORA_OFF] : 1);
    if (!off) return ORA_E_NOMEM;
    if ((rc = stream_decode(&r, ORA_OFF, off)) != ORA_OK) { free(off); return rc; }
    uint32_t e = 0, sum_lit = 0, sum_all = 0;
    for (uint32_t q = 0; q < r.n_seq; q++) {
        uint32_t ll = len[2 * q], ml = len[2 * q + 1];
        if (ll == 255) { if (e >= r.n_extras) { rc = ORA_E_CORRUPT; break; } ll = rd16(r.extras + 2 * (size_t)e++); }
        if (ml == 255) { if (e >= r.n_extras) { rc = ORA_E_CORRUPT; break; } ml = rd16(r.extras + 2 * (size_t)e++); }
        t->lit_len[q] = ll;
        t->match_len[q] = ml + 4;
        uint64_t src = 0;
        for (uint32_t j = 0; j < r.off_nbytes; j++) src |= (uint64_t)off[q * r.off_nbytes + j] << (8 * j);
        t->src[q] = src;
        t->tag[q] = (r.tags[q >> 1] >> ((q & 1) * 4)) & 15u;
        sum_lit += ll;
        sum_all += ll + ml + 4;
        if (sum_lit > r.n_lit || sum_all > r.block_len) { rc = ORA_E_CORRUPT; break; }
    }
    free(off);
    if (rc != ORA_OK) return rc;
    if (e != r.n_extras) return ORA_E_CORRUPT;
    t->trailing = r.n_lit - sum_lit;
    if (sum_all + t->trailing != r.block_len) return ORA_E_CORRUPT;
    return ORA_OK;
}

int ora_decode_tokens(const uint8_t *c, size_t clen, uint64_t block, uint32_t *n_seq,
                      uint32_t *lit_len, uint32_t *match_len, uint64_t *src, uint8_t *tags)
{
    ora_container k;
    int rc = ora_container_open(c, clen, &k);
    if (rc != ORA_OK) return rc;
    ora_tokens *t = (ora_tokens *)malloc(sizeof *t);
    if (!t) return ORA_E_NOMEM;
    rc = ora_tokens_decode(&k, block, t);
    if (rc == ORA_OK) {
        *n_seq = t->n_seq;
        for (uint32_t q = 0; q < t->n_seq; q++) {
            if (lit_len) lit_len[q] = t->lit_len[q];
            if (match_len) match_len[q] = t->match_len[q];
            if (src) src[q] = t->src[q];
            if (tags) tags[q] = t->tag[q];
        }
    }
    free(t);
    return rc;
}

/* ---------------------------------------------------------------- decoder #1 */

/* decoder #1 step 2.4: emit one block from its tokens (literal run, then memcpy from the absolute position) */
static int emit_block(const ora_tokens *t, uint64_t b, uint8_t *out)
{
    uint64_t pos = b * ORA_B, end = pos + t->block_len;
    uint32_t lp = 0;
    for (uint32_t q = 0; q < t->n_seq; q++) {
        memcpy(out + pos, t->lit + lp, t->lit_len[q]);           /* literal run */
        pos += t->lit_len[q]; lp += t->lit_len[q];
        uint64_t src = t->src[q], ml = t->match_len[q];
        if (src + ml > pos || pos + ml > end) return ORA_E_CORRUPT; /* strictly before */
        memcpy(out + pos, out + src, ml);                         /* absolute-offset copy */
        pos += ml;
    }
    memcpy(out + pos, t->lit + lp, t->trailing);
    pos += t->trailing; lp += t->trailing;
    if (lp != t->n_lit || pos != end) return ORA_E_CORRUPT;
    return ORA_OK;
}

int ora_decode_all(const uint8_t *c, size_t clen, uint8_t *out, size_t cap)
{
    ora_container k;
    int rc = ora_container_open(c, clen, &k);
    if (rc != ORA_OK) return rc;
    if (cap < k.info.total_len) return ORA_E_CAPACITY;
    ora_tokens *t = (ora_tokens *)malloc(sizeof *t);
    if (!t) return ORA_E_NOMEM;
    for (uint64_t b = 0; b < k.info.n_blocks && rc == ORA_OK; b++) {
        if ((rc = ora_tokens_decode(&k, b, t)) != ORA_OK) break;
        rc = emit_block(t, b, out);
    }
    free(t);
    return rc;
}

/* Decoder #1 with the entropy stage spread over host threads (SURVEY.md section 8d "oracle timed beside it",
 * variant b): blocks are independent in the entropy layer, so groups of blocks are entropy-decoded
 * and parsed in parallel (the same ora_tokens_decode per block); the match stage then emits them one after the
 * other in block order, because a copy may read any earlier output byte. Same result as
 * ora_decode_all by construction; pinned by tests/test_oracle_codec.py. */
int ora_decode_all_mt(const uint8_t *c, size_t clen, uint8_t *out, size_t cap, uint32_t threads)
{
    ora_container k;
    int rc = ora_container_open(c, clen, &k);
    if (rc != ORA_OK) return rc;
    if (cap < k.info.total_len) return ORA_E_CAPACITY;
    if (threads < 1) threads = 1;
    const uint64_t group = 4 * (uint64_t)threads;
    ora_tokens *t = (ora_tokens *)malloc(sizeof *t * group);
    int *rcs = (int *)malloc(sizeof *rcs * group);
    if (!t || !rcs) { free(t); free(rcs); return ORA_E_NOMEM; }
    for (uint64_t b0 = 0; b0 < k.info.n_blocks && rc == ORA_OK; b0 += group) {
        const uint64_t n = k.info.n_blocks - b0 < group ? k.info.n_blocks - b0 : group;
#pragma omp parallel for schedule(dynamic, 1) num_threads(threads)
        for (int64_t i = 0; i < (int64_t)n; i++) rcs[i] = ora_tokens_decode(&k, b0 + (uint64_t)i, &t[i]);
        for (uint64_t i = 0; i < n && rc == ORA_OK; i++) {
            rc = rcs[i];
            if (rc == ORA_OK) rc = emit_block(&t[i], b0 + i, out);
        }
    }
    free(t); free(rcs);
    return rc;
}

/* ---------------------------------------------------------------- decoder #2 */

/* memoised per-block token view for the origin chase */
typedef struct {
    uint32_t n_seq, block_len;
    uint32_t *seq_start; /* n_seq+1: output offset (in block) where sequence q's literal run starts;
                            entry n_seq = start of the trailing literals */
    uint32_t *dst;       /* n_seq: output offset (in block) of match q */
    uint32_t *lit_pos;   /* n_seq+1: index into lit[] of sequence q's first literal */
    uint64_t *src;       /* n_seq */
    uint8_t *lit;        /* n_lit */
} iso_block;

struct ora_iso {
    ora_container k;
    iso_block **cache; /* n_blocks */
};

int ora_iso_open(const uint8_t *c, size_t clen, ora_iso **out)
{
    ora_iso *x = (ora_iso *)calloc(1, sizeof *x);
    if (!x) return ORA_E_NOMEM;
    int rc = ora_container_open(c, clen, &x->k);
    if (rc != ORA_OK) { free(x); return rc; }
    x->cache = (iso_block **)calloc(x->k.info.n_blocks ? x->k.info.n_blocks : 1, sizeof(iso_block *));
    if (!x->cache) { free(x); return ORA_E_NOMEM; }
    *out = x;
    return ORA_OK;
}

static void iso_block_free(iso_block *ib)
{
    if (!ib) return;
    free(ib->seq_start); free(ib->dst); free(ib->lit_pos); free(ib->src); free(ib->lit); free(ib);
}

void ora_iso_close(ora_iso *x)
{
    if (!x) return;
    for (uint64_t b = 0; b < x->k.info.n_blocks; b++) iso_block_free(x->cache[b]);
    free(x->cache);
    free(x);
}

static int iso_get(ora_iso *x, uint64_t b, iso_block **out)
{
    if (x->cache[b]) { *out = x->cache[b]; return ORA_OK; }
    ora_tokens *t = (ora_tokens *)malloc(sizeof *t);
    if (!t) return ORA_E_NOMEM;
    int rc = ora_tokens_decode(&x->k, b, t);
    if (rc != ORA_OK) { free(t); return rc; }
    iso_block *ib = (iso_block *)calloc(1, sizeof *ib);
    uint32_t n = t->n_seq;
    ib->n_seq = n; ib->block_len = t->block_len;
    ib->seq_start = (uint32_t *)malloc(sizeof(uint32_t) * (n + 1));
    ib->dst = (uint32_t *)malloc(sizeof(uint32_t) * (n + 1));
    ib->lit_pos = (uint32_t *)malloc(sizeof(uint32_t) * (n + 1));
    ib->src = (uint64_t *)malloc(sizeof(uint64_t) * (n + 1));
    ib->lit = (uint8_t *)malloc(t->n_lit ? t->n_lit : 1);
    memcpy(ib->lit, t->lit, t->n_lit);
    uint32_t pos = 0, lp = 0;
    for (uint32_t q = 0; q < n; q++) {
        ib->seq_start[q] = pos; ib->lit_pos[q] = lp;
        pos += t->lit_len[q]; lp += t->lit_len[q];
        ib->dst[q] = pos; ib->src[q] = t->src[q];
        if (t->src[q] + t->match_len[q] > b * ORA_B + pos) rc = ORA_E_CORRUPT; /* src+len <= dst */
        pos += t->match_len[q];
    }
    ib->seq_start[n] = pos; ib->lit_pos[n] = lp;
    free(t);
    if (rc != ORA_OK) { iso_block_free(ib); return rc; }
    x->cache[b] = ib;
    *out = ib;
    return ORA_OK;
}

/* the byte at absolute position p, by chasing its origin through the compressed data */
static int iso_byte(ora_iso *x, uint64_t p, uint8_t *byte, uint32_t *hops)
{
    uint32_t h = 0;
    for (;;) {
        uint64_t b = p >> ORA_BLOG;
        uint32_t o = (uint32_t)(p & (ORA_B - 1));
        iso_block *ib;
        int rc = iso_get(x, b, &ib);
        if (rc != ORA_OK) return rc;
        if (o >= ib->block_len) return ORA_E_CORRUPT;
        /* the sequence q with seq_start[q] <= o < seq_start[q+1]; q == n_seq: trailing literals */
        uint32_t lo = 0, hi = ib->n_seq; /* invariant: seq_start[lo] <= o */
        while (lo < hi) {
            uint32_t mid = (lo + hi + 1) / 2;
            if (ib->seq_start[mid] <= o) lo = mid; else hi = mid - 1;
        }
        uint32_t q = lo;
        if (q == ib->n_seq || o < ib->dst[q]) {          /* a literal: the origin */
            *byte = ib->lit[ib->lit_pos[q] + (o - ib->seq_start[q])];
            *hops = h;
            return ORA_OK;
        }
        uint64_t nxt = ib->src[q] + (o - ib->dst[q]);    /* a match: follow the absolute offset */
        if (nxt >= p) return ORA_E_CORRUPT;              /* strictly before: the chase terminates */
        p = nxt;
        h++;
    }
}

int ora_iso_decode(ora_iso *x, uint64_t block, uint8_t *dst, size_t cap, uint32_t *block_len,
                   uint32_t *max_hops)
{
    if (!x || !dst) return ORA_E_ARG;
    if (block >= x->k.info.n_blocks) return ORA_E_RANGE;
    iso_block *ib;
    int rc = iso_get(x, block, &ib);
    if (rc != ORA_OK) return rc;
    if (cap < ib->block_len) return ORA_E_CAPACITY;
    uint32_t mh = 0, len = ib->block_len;
    for (uint32_t o = 0; o < len; o++) {
        uint32_t h;
        if ((rc = iso_byte(x, block * ORA_B + o, dst + o, &h)) != ORA_OK) return rc;
        if (h > mh) mh = h;
    }
    if (block_len) *block_len = len;
    if (max_hops) *max_hops = mh;
    return ORA_OK;
}

/* ---------------------------------------------------------------- validator */

int ora_validate(const uint8_t *c, size_t clen, ora_validate_report *rep)
{
    ora_container k;
    int rc = ora_container_open(c, clen, &k);
    if (rc != ORA_OK) return rc;
    ora_validate_report R;
    memset(&R, 0, sizeof R);
    R.min_match_seen = 0xFFFFFFFFu;
    uint64_t n = k.info.total_len;
    uint8_t *depth = (uint8_t *)calloc(n ? n : 1, 1);   /* copy-hop depth of every byte, saturating */
    uint8_t *level = (uint8_t *)malloc(ORA_B);          /* in-block tag of the match that wrote a byte */
    ora_tokens *t = (ora_tokens *)malloc(sizeof *t);
    uint64_t *seen = (uint64_t *)calloc((k.info.n_blocks + 63) / 64 + 1, 8);
    if (!depth || !level || !t || !seen) { free(depth); free(level); free(t); free(seen); return ORA_E_NOMEM; }
    int promise_broken = 0;
    double sum_src_blocks = 0;
    for (uint64_t b = 0; b < k.info.n_blocks && rc == ORA_OK; b++) {
        if ((rc = ora_tokens_decode(&k, b, t)) != ORA_OK) break;
        uint64_t start = b * ORA_B, pos = start, end = start + t->block_len;
        memset(level, 0, ORA_B);
        uint32_t n_src_blocks = 0;
        uint64_t touched[ORA_MAX_SEQ * 2]; uint32_t n_touched = 0;
        for (uint32_t q = 0; q < t->n_seq; q++) {
            pos += t->lit_len[q];
            uint64_t src = t->src[q], ml = t->match_len[q];
            if (ml < 4 || src + ml > pos || pos + ml > end) { rc = ORA_E_CORRUPT; break; }
            if (ml < R.min_match_seen) R.min_match_seen = (uint32_t)ml;
            uint32_t d = 0, lv = 0;
            for (uint64_t j = 0; j < ml; j++) {
                if (depth[src + j] > d) d = depth[src + j];
                if (src + j >= start && level[src + j - start] + 1u > lv) lv = level[src + j - start] + 1u;
            }
            if (src + ml > start && lv == 0) lv = 1; /* touches the block through literal bytes only */
            d = d + 1 > 255 ? 255 : d + 1;
            if (lv != t->tag[q] || lv > 15) promise_broken = 1;
            if (src + ml <= start) R.n_matches_cross++;
            else if (src >= start) R.n_matches_intra++;
            else R.n_matches_spanning++;
            if (k.info.window) {
                uint64_t last_blk = (src + ml - 1) >> ORA_BLOG;
                int inside = src >= start;
                int old = last_blk + k.info.window <= b;
                if (!inside && !old) promise_broken = 1;
            }
            for (uint64_t sb = src >> ORA_BLOG; sb <= ((src + ml - 1) >> ORA_BLOG); sb++) {
                if (sb == b) continue;
                if (!(seen[sb >> 6] >> (sb & 63) & 1)) { seen[sb >> 6] |= (uint64_t)1 << (sb & 63); touched[n_touched++] = sb; n_src_blocks++; }
            }
            for (uint64_t j = 0; j < ml; j++) { depth[pos + j] = (uint8_t)d; level[pos + j - start] = (uint8_t)lv; }
            if (d > R.max_depth_seen) R.max_depth_seen = d;
            if (lv > R.max_level_seen) R.max_level_seen = lv;
            pos += ml;
            R.n_seq++;
        }
        for (uint32_t i = 0; i < n_touched; i++) seen[touched[i] >> 6] &= ~((uint64_t)1 << (touched[i] & 63));
        if (n_src_blocks > R.max_src_blocks_per_block) R.max_src_blocks_per_block = n_src_blocks;
        if (k.info.max_fanout && n_src_blocks > k.info.max_fanout) promise_broken = 1;
        sum_src_blocks += n_src_blocks;
    }
    if (rc == ORA_OK) {
        if (k.info.max_depth && R.max_depth_seen > k.info.max_depth) promise_broken = 1;
        if (R.max_level_seen > k.info.max_level) promise_broken = 1;
        R.mean_src_blocks_per_block = k.info.n_blocks ? sum_src_blocks / (double)k.info.n_blocks : 0.0;
        if (R.min_match_seen == 0xFFFFFFFFu) R.min_match_seen = 0;
        if (rep) *rep = R;
        if (promise_broken) rc = ORA_E_PROMISE;
    }
    free(depth); free(level); free(t); free(seen);
    return rc;
}
