/* ORACLE (test infrastructure) — the CPU encoder.
 *
 * "The encoder performs a global match search and partitions output into fixed-size
 * blocks"; every back-reference is an absolute position in the decompressed output.
 * BASELINE.json north_star: greedy hash-chain global match search, min match 4, absolute offsets,
 * every reference strictly before its own position. The paper gives no further encoder detail
 * (its Paper 1 is not in the container); readings A14-A16 list the choices made here.
 * Many encodings of one input are valid: parity is never judged on compressed bytes, only on
 * decoded bytes (reading A19). The encoder is deterministic and independent of `threads`.
 *
 * Definition (sequential semantics):
 *   Blocks are parsed in batches of `batch` consecutive blocks (1 when R == 0). Before a batch
 *   starting at block s, every position of blocks <= s-R (R > 0) resp. < s (R == 0) is appended
 *   to the global hash chains, in increasing position order. Inside block b at position i, with
 *   at least T bytes left in the block, candidates are tried newest-first: up to chain_depth from
 *   the block's own chain, then up to chain_depth from the global chain. A candidate j yields
 *   the longest l with in[j..j+l) == in[i..i+l), l <= block_end - i, l <= i - j (src+len <= dst),
 *   j+l <= end of eligible region (R > 0, global candidates), every source byte of copy depth
 *   < D (D > 0) and, inside the block, of tag < max_level. The longest wins, the first found
 *   among equals; it is accepted if l >= T. Otherwise in[i] is a literal.
 *   long_hash > 0 (SURVEY.md reading A14: "4-byte hash + optional 12-byte long hash; chain depth 32
 *   (+16 long)"): a second global table keyed on long_hash bytes is probed first, up to long_chain
 *   candidates, newest first, under the same limits; then the chains above.
 *   max_fanout F > 0 (seek-aware policy; a seek needs every block
 *   a block copies from): the matches of one block read from at most F distinct earlier blocks. A global
 *   candidate whose first source block is neither used yet nor affordable is skipped; one that runs on
 *   into a second block that is neither is cut at the block boundary.
 *   max_seq > 0: a block holds at most max_seq sequences; once it has that many, the rest of the block is
 *   literals (a decoder sizes its per-block tables for the densest block of a container).
 */
#include "container.h"

#include <stdlib.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define LOCAL_HASH_BITS 13
#define NONE16 0xFFFFu

typedef struct {
    uint32_t lit_len, match_len;
    uint64_t src;
    uint8_t tag;
} enc_seq;

typedef struct {
    uint8_t *rec;          /* serialised record */
    size_t rec_bytes;
    uint32_t states[3][32];
    ora_enc_stats st;
} enc_block;

typedef struct {
    uint16_t lhead[1u << LOCAL_HASH_BITS];
    uint16_t lprev[ORA_B];
    uint8_t level[ORA_B];
    enc_seq seq[ORA_MAX_SEQ];
    uint8_t lit[ORA_B];
    uint8_t len_sym[2 * ORA_MAX_SEQ];
    uint8_t off_sym[8 * ORA_MAX_SEQ];
    uint16_t extras[2 * ORA_MAX_SEQ];
    uint16_t words[3][8 * ORA_MAX_SEQ];
    uint64_t *fan_bits;    /* max_fanout: bitmap over blocks, the source blocks this block uses */
    uint32_t fan_list[2 * ORA_MAX_SEQ], fan_n;
} enc_scratch;

typedef struct {
    const uint8_t *in;
    size_t n;
    ora_enc_params p;
    uint32_t hash_bytes, hash_bits;
    uint32_t *head;  /* position+1 of the newest inserted position per hash, 0 = empty */
    uint32_t *prev;  /* position+1 of the previous position with the same hash */
    uint8_t *depth;  /* copy-hop depth of every parsed byte (saturating at 255) */
    uint32_t long_bits;
    uint32_t *head2; /* long hash: same scheme, keyed on p.long_hash bytes */
    uint32_t *prev2;
} enc_ctx;

int ora_block_log2(void) { return ORA_BLOG; }

void ora_enc_params_default(ora_enc_params *p)
{
    p->min_match = 4;
    p->chain_depth = 32;
    p->max_depth = 0;
    p->window = 0;
    p->max_level = 15;
    p->offset_width = 4;
    p->threads = 1;
    p->batch = 64;
    p->raw_slack_pct = 0;
    p->max_fanout = 0;
    p->long_hash = 0;
    p->long_chain = 16;
    p->max_seq = 0;
}

size_t ora_encode_bound(size_t n)
{
    size_t nb = (n + ORA_B - 1) / ORA_B;
    /* per block: index entry, record header, 3 tables, section padding, and at worst
     * ~1.01 x 16-bit words per byte-symbol plus token overhead */
    return ORA_HDR_BYTES + 16 + (nb + 1) * 8 + nb * (384 + 32 + 3 * (32 + 512) + 8 * 16) + 3 * n + 4096;
}

static inline uint32_t hash_at(const enc_ctx *e, size_t i)
{
    uint64_t v = 0;
    memcpy(&v, e->in + i, e->hash_bytes); /* little-endian hosts only (oracle runs on x86-64) */
    return (uint32_t)((v * 0x9E3779B97F4A7C15ull) >> (64 - e->hash_bits));
}

static inline uint32_t long_hash_at(const enc_ctx *e, size_t i)
{
    uint64_t a = 0, b = 0;
    const uint32_t nb = e->p.long_hash;          /* 9..16 */
    memcpy(&a, e->in + i, 8);
    memcpy(&b, e->in + i + 8, nb - 8);
    return (uint32_t)(((a * 0x9E3779B97F4A7C15ull) ^ (b * 0xC2B2AE3D27D4EB4Full)) * 0x9E3779B97F4A7C15ull >> (64 - e->long_bits));
}

static void global_insert(enc_ctx *e, size_t from, size_t to)
{
    for (size_t p = from; p < to; p++) {
        if (p + e->hash_bytes > e->n) break;
        if (e->p.max_depth && e->depth[p] >= e->p.max_depth) continue;
        uint32_t h = hash_at(e, p);
        e->prev[p] = e->head[h];
        e->head[h] = (uint32_t)p + 1;
        if (e->head2 && p + e->p.long_hash <= e->n) {
            uint32_t h2 = long_hash_at(e, p);
            e->prev2[p] = e->head2[h2];
            e->head2[h2] = (uint32_t)p + 1;
        }
    }
}

/* max_fanout: how far a global candidate at j may run, given the source blocks the block already uses */
static inline int fan_has(const enc_scratch *s, uint64_t blk) { return (int)(s->fan_bits[blk >> 6] >> (blk & 63) & 1); }
static inline uint32_t fan_limit(const enc_ctx *e, const enc_scratch *s, size_t j, uint32_t maxlen)
{
    const uint32_t F = e->p.max_fanout;
    if (!F) return maxlen;
    const uint64_t b0 = j >> ORA_BLOG;
    uint32_t room = F - s->fan_n;
    if (!fan_has(s, b0)) { if (!room) return 0; room--; }
    const size_t to_end = ((size_t)(b0 + 1) << ORA_BLOG) - j;      /* bytes left in block b0 */
    if (maxlen > to_end && !fan_has(s, b0 + 1) && !room) maxlen = (uint32_t)to_end;
    return maxlen;
}
static inline void fan_add(enc_scratch *s, uint64_t blk)
{
    if (fan_has(s, blk)) return;
    s->fan_bits[blk >> 6] |= (uint64_t)1 << (blk & 63);
    s->fan_list[s->fan_n++] = (uint32_t)blk;
}

/* candidate j for position i: common prefix under all limits of the definition above */
static inline uint32_t try_candidate(const enc_ctx *e, const uint8_t *level, size_t B0, size_t i,
                                     size_t j, uint32_t maxlen, uint32_t best)
{
    const uint8_t *in = e->in;
    if (maxlen <= best) return 0;
    if (in[j + best] != in[i + best]) return 0;
    uint32_t l = 0, D = e->p.max_depth, L = e->p.max_level;
    while (l < maxlen && in[j + l] == in[i + l]) {
        if (D && e->depth[j + l] >= D) break;
        if (j + l >= B0 && level[j + l - B0] >= L) break;
        l++;
    }
    return l;
}

static void parse_block(enc_ctx *e, uint64_t b, size_t elig_end, enc_scratch *s, uint32_t *n_seq_out,
                        uint32_t *n_lit_out, ora_enc_stats *st)
{
    const uint8_t *in = e->in;
    const size_t B0 = (size_t)b * ORA_B;
    const size_t B1 = (B0 + ORA_B < e->n) ? B0 + ORA_B : e->n;
    const uint32_t T = e->p.min_match, chain = e->p.chain_depth, D = e->p.max_depth, L = e->p.max_level;
    const uint32_t lmask = (1u << LOCAL_HASH_BITS) - 1;
    const uint32_t max_seq = e->p.max_seq && e->p.max_seq < ORA_MAX_SEQ ? e->p.max_seq : ORA_MAX_SEQ;
    uint32_t n_seq = 0, n_lit = 0;
    size_t lit_start = B0, i = B0;
    memset(s->lhead, 0xFF, sizeof s->lhead);
    memset(s->level, 0, sizeof s->level);
    s->fan_n = 0;

    while (i < B1) {
        uint32_t best = 0;
        size_t best_src = 0;
        const uint32_t remaining = (uint32_t)(B1 - i);
        const int can_hash = i + e->hash_bytes <= e->n;
        uint32_t h = 0;
        if (can_hash) h = hash_at(e, i);
        if (can_hash && remaining >= T && n_seq < max_seq) {
            /* the block's own chain, newest first */
            uint32_t cand = s->lhead[h & lmask];
            for (uint32_t steps = 0; cand != NONE16 && steps < chain; steps++, cand = s->lprev[cand]) {
                size_t j = B0 + cand;
                uint32_t maxlen = remaining;
                if (i - j < maxlen) maxlen = (uint32_t)(i - j);
                uint32_t l = try_candidate(e, s->level, B0, i, j, maxlen, best);
                if (l > best) { best = l; best_src = j; }
            }
            /* the long-hash global chain, newest first */
            if (e->head2 && i + e->p.long_hash <= e->n) {
                uint32_t g = e->head2[long_hash_at(e, i)];
                for (uint32_t steps = 0; g != 0 && steps < e->p.long_chain; steps++, g = e->prev2[g - 1]) {
                    size_t j = g - 1;
                    uint32_t maxlen = remaining;
                    if (i - j < maxlen) maxlen = (uint32_t)(i - j);
                    if (e->p.window && elig_end - j < maxlen) maxlen = (uint32_t)(elig_end - j);
                    maxlen = fan_limit(e, s, j, maxlen);
                    uint32_t l = try_candidate(e, s->level, B0, i, j, maxlen, best);
                    if (l > best) { best = l; best_src = j; }
                }
            }
            /* the global chain, newest first */
            uint32_t g = e->head[h];
            for (uint32_t steps = 0; g != 0 && steps < chain; steps++, g = e->prev[g - 1]) {
                size_t j = g - 1;
                uint32_t maxlen = remaining;
                if (i - j < maxlen) maxlen = (uint32_t)(i - j);
                if (e->p.window && elig_end - j < maxlen) maxlen = (uint32_t)(elig_end - j);
                maxlen = fan_limit(e, s, j, maxlen);
                uint32_t l = try_candidate(e, s->level, B0, i, j, maxlen, best);
                if (l > best) { best = l; best_src = j; }
            }
        }
        if (best >= T && best >= 4) {
            enc_seq *q = &s->seq[n_seq++];
            q->lit_len = (uint32_t)(i - lit_start);
            q->match_len = best;
            q->src = best_src;
            memcpy(s->lit + n_lit, in + lit_start, q->lit_len);
            n_lit += q->lit_len;
            uint32_t d = 0, lv = 0;
            for (uint32_t l = 0; l < best; l++) {
                if (e->depth[best_src + l] > d) d = e->depth[best_src + l];
                if (best_src + l >= B0 && s->level[best_src + l - B0] + 1u > lv) lv = s->level[best_src + l - B0] + 1u;
            }
            d = d + 1 > 255 ? 255 : d + 1;
            q->tag = (uint8_t)lv;
            if (e->p.max_fanout && best_src < B0) {
                fan_add(s, best_src >> ORA_BLOG);
                const uint64_t lastb = (best_src + best - 1) >> ORA_BLOG;
                if (lastb < b) fan_add(s, lastb);
            }
            if (d > st->max_depth_seen) st->max_depth_seen = d;
            if (lv > st->max_level_seen) st->max_level_seen = lv;
            st->match_bytes += best;
            if (best_src + best > B0) st->intra_match_bytes += best;
            for (uint32_t l = 0; l < best; l++) {
                size_t p = i + l;
                e->depth[p] = (uint8_t)d;
                s->level[p - B0] = (uint8_t)lv;
                if (p + e->hash_bytes <= e->n && lv < L && !(D && d >= D)) {
                    uint32_t hp = hash_at(e, p) & lmask;
                    s->lprev[p - B0] = s->lhead[hp];
                    s->lhead[hp] = (uint16_t)(p - B0);
                }
            }
            i += best;
            lit_start = i;
        } else {
            e->depth[i] = 0;
            if (can_hash) {
                s->lprev[i - B0] = s->lhead[h & lmask];
                s->lhead[h & lmask] = (uint16_t)(i - B0);
            }
            i++;
        }
    }
    for (uint32_t k = 0; k < s->fan_n; k++) s->fan_bits[s->fan_list[k] >> 6] = 0;
    memcpy(s->lit + n_lit, in + lit_start, B1 - lit_start); /* trailing literals */
    n_lit += (uint32_t)(B1 - lit_start);
    *n_seq_out = n_seq;
    *n_lit_out = n_lit;
}

/* FORMAT.md section 3 "Table": bitmap + u16 freq per present symbol */
static uint32_t table_write(uint8_t *dst, const uint16_t freq[256])
{
    uint32_t np = 0;
    memset(dst, 0, 32);
    for (int s = 0; s < 256; s++) {
        if (!freq[s]) continue;
        dst[s >> 3] |= (uint8_t)(1u << (s & 7));
        wr16(dst + 32 + 2 * np, freq[s]);
        np++;
    }
    return 32 + 2 * np;
}

/* FORMAT.md sections 2-4: streams, tables, rANS, record layout */
static int serialise_block(const enc_ctx *e, uint64_t b, enc_scratch *s, uint32_t n_seq, uint32_t n_lit,
                           enc_block *out)
{
    uint32_t n_extras = 0, off_nbytes = 1;
    uint64_t max_src = 0;
    for (uint32_t q = 0; q < n_seq; q++) if (s->seq[q].src > max_src) max_src = s->seq[q].src;
    while (off_nbytes < 8 && (max_src >> (8 * off_nbytes)) != 0) off_nbytes++;
    if (off_nbytes > e->p.offset_width) return ORA_E_ARG;
    for (uint32_t q = 0; q < n_seq; q++) {
        const enc_seq *t = &s->seq[q];
        uint32_t ll = t->lit_len, ml = t->match_len - 4;
        s->len_sym[2 * q] = (uint8_t)(ll < 255 ? ll : 255);
        if (ll >= 255) s->extras[n_extras++] = (uint16_t)ll;
        s->len_sym[2 * q + 1] = (uint8_t)(ml < 255 ? ml : 255);
        if (ml >= 255) s->extras[n_extras++] = (uint16_t)ml;
        for (uint32_t j = 0; j < off_nbytes; j++) s->off_sym[q * off_nbytes + j] = (uint8_t)(t->src >> (8 * j));
    }
    const uint8_t *sym[3] = { s->lit, s->len_sym, s->off_sym };
    uint32_t n_sym[3] = { n_lit, 2 * n_seq, off_nbytes * n_seq };
    uint8_t tables[3][32 + 512];
    uint32_t tbl_bytes[3] = { 0, 0, 0 };
    size_t n_words[3] = { 0, 0, 0 };
    uint32_t modes = 0;
    for (int k = 0; k < 3; k++) {
        uint32_t count[256] = { 0 };
        uint16_t freq[256];
        for (uint32_t i = 0; i < n_sym[k]; i++) count[sym[k][i]]++;
        ora_quantise(count, freq);
        int rc = ora_rans_encode(sym[k], n_sym[k], freq, 32, out->states[k], s->words[k], &n_words[k]);
        if (rc != ORA_OK) return rc;
        if (n_sym[k]) tbl_bytes[k] = table_write(tables[k], freq);
        /* selective entropy ("apply ANS selectively"; FORMAT.md section 2 modes): a stream of one
         * repeated symbol is stored as that symbol (CONST); otherwise keep the stream verbatim (RAW) when rANS does
         * not pay for itself */
        if (n_sym[k] && e->p.raw_slack_pct != 0xFFFFFFFFu && count[sym[k][0]] == n_sym[k]) {
            modes |= 2u << (2 * k);
            tbl_bytes[k] = 0;
            n_words[k] = 1;
            s->words[k][0] = sym[k][0];
            for (int l = 0; l < 32; l++) out->states[k][l] = 65536u;
            out->st.n_const[k]++;
        } else if (n_sym[k] && e->p.raw_slack_pct != 0xFFFFFFFFu &&
            (uint64_t)n_sym[k] * 100 <= ((uint64_t)tbl_bytes[k] + 2 * (uint64_t)n_words[k]) * (100 + (uint64_t)e->p.raw_slack_pct)) {
            modes |= 1u << (2 * k);
            tbl_bytes[k] = 0;
            n_words[k] = (n_sym[k] + 1) / 2;
            for (uint32_t i = 0; i < n_words[k]; i++) {
                uint32_t lo = sym[k][2 * i], hi = 2 * i + 1 < n_sym[k] ? sym[k][2 * i + 1] : 0;
                s->words[k][i] = (uint16_t)(lo | hi << 8);            /* bytes in order, little-endian words */
            }
            for (int l = 0; l < 32; l++) out->states[k][l] = 65536u;
            out->st.n_raw[k]++;
        }
    }
    size_t pos = ORA_REC_HDR_BYTES;
    for (int k = 0; k < 3; k++) pos = pad16(pos) + tbl_bytes[k];
    pos = pad16(pos) + 2 * (size_t)n_extras;
    pos = pad16(pos) + (n_seq + 1) / 2;
    for (int k = 0; k < 3; k++) pos = pad16(pos) + 2 * n_words[k];
    size_t rec_bytes = pad16(pos);
    uint8_t *rec = (uint8_t *)calloc(rec_bytes, 1);
    if (!rec) return ORA_E_NOMEM;
    wr16(rec + 0, n_seq); wr16(rec + 2, n_lit); wr16(rec + 4, n_extras);
    rec[6] = (uint8_t)off_nbytes; rec[7] = (uint8_t)modes;
    for (int k = 0; k < 3; k++) { wr32(rec + 8 + 4 * k, (uint32_t)n_words[k]); wr16(rec + 20 + 2 * k, tbl_bytes[k]); }
    pos = ORA_REC_HDR_BYTES;
    for (int k = 0; k < 3; k++) { pos = pad16(pos); memcpy(rec + pos, tables[k], tbl_bytes[k]); pos += tbl_bytes[k]; }
    pos = pad16(pos);
    for (uint32_t i = 0; i < n_extras; i++) wr16(rec + pos + 2 * (size_t)i, s->extras[i]);
    pos += 2 * (size_t)n_extras;
    pos = pad16(pos);
    for (uint32_t q = 0; q < n_seq; q++) rec[pos + (q >> 1)] |= (uint8_t)((s->seq[q].tag & 15u) << ((q & 1) * 4));
    pos += (n_seq + 1) / 2;
    for (int k = 0; k < 3; k++) {
        pos = pad16(pos);
        for (size_t i = 0; i < n_words[k]; i++) wr16(rec + pos + 2 * i, s->words[k][i]);
        pos += 2 * n_words[k];
    }
    out->rec = rec;
    out->rec_bytes = rec_bytes;
    out->st.n_seq += n_seq; out->st.n_lit += n_lit; out->st.n_extras += n_extras;
    for (int k = 0; k < 3; k++) { out->st.n_sym[k] += n_sym[k]; out->st.n_words[k] += n_words[k]; out->st.table_bytes += tbl_bytes[k]; }
    (void)b;
    return ORA_OK;
}

int ora_encode(const uint8_t *in, size_t n, const ora_enc_params *pp, uint8_t *out, size_t cap,
               size_t *out_len, ora_enc_stats *stats)
{
    if ((!in && n) || !pp || !out || !out_len) return ORA_E_ARG;
    enc_ctx e;
    memset(&e, 0, sizeof e);
    e.in = in; e.n = n; e.p = *pp;
    if (e.p.min_match < 4 || e.p.chain_depth < 1) return ORA_E_ARG;
    if (e.p.max_level < 1 || e.p.max_level > 15) return ORA_E_ARG;
    if (e.p.offset_width != 4 && e.p.offset_width != 8) return ORA_E_ARG;
    if (n >= 0xFFFFFFF0ull) return ORA_E_ARG;          /* oracle limit (u32 chains), not a format limit */
    if (e.p.offset_width == 4 && n > 0xFFFFFFFFull) return ORA_E_ARG;
    if (e.p.max_depth > 254) return ORA_E_ARG;
    if (e.p.max_fanout > 0xFFFF || e.p.min_match > 0xFFFF) return ORA_E_ARG;
    if (e.p.long_hash && (e.p.long_hash < 9 || e.p.long_hash > 16 || e.p.long_chain < 1)) return ORA_E_ARG;
    if (e.p.threads < 1) e.p.threads = 1;
    if (e.p.batch < 1) e.p.batch = 1;
    e.hash_bytes = e.p.min_match < 8 ? e.p.min_match : 8;
    e.hash_bits = 16;
    while (e.hash_bits < 24 && ((size_t)1 << (e.hash_bits + 2)) < n) e.hash_bits++;

    const uint64_t nb = (n + ORA_B - 1) / ORA_B;
    const uint64_t R = e.p.window;
    const uint64_t P = R ? e.p.batch : 1;
    int rc = ORA_OK;
    enc_block *blocks = (enc_block *)calloc(nb ? nb : 1, sizeof(enc_block));
    enc_scratch *scr = (enc_scratch *)malloc(sizeof(enc_scratch) * e.p.threads);
    e.head = (uint32_t *)calloc((size_t)1 << e.hash_bits, sizeof(uint32_t));
    e.prev = (uint32_t *)malloc(sizeof(uint32_t) * (n ? n : 1));
    e.depth = (uint8_t *)calloc(n ? n : 1, 1);
    if (!blocks || !scr || !e.head || !e.prev || !e.depth) { rc = ORA_E_NOMEM; goto done; }
    for (uint32_t t = 0; t < e.p.threads; t++) scr[t].fan_bits = NULL;
    for (uint32_t t = 0; t < e.p.threads; t++) {
        scr[t].fan_bits = (uint64_t *)calloc((size_t)(nb / 64 + 2), 8);
        if (!scr[t].fan_bits) { rc = ORA_E_NOMEM; goto done; }
    }
    if (e.p.long_hash) {
        e.long_bits = e.hash_bits;
        e.head2 = (uint32_t *)calloc((size_t)1 << e.long_bits, sizeof(uint32_t));
        e.prev2 = (uint32_t *)malloc(sizeof(uint32_t) * (n ? n : 1));
        if (!e.head2 || !e.prev2) { rc = ORA_E_NOMEM; goto done; }
    }

    size_t inserted = 0;
    for (uint64_t s = 0; s < nb && rc == ORA_OK; s += P) {
        uint64_t s_end = s + P < nb ? s + P : nb;
        size_t elig_end;
        if (R) elig_end = (s + 1 > R) ? (size_t)(s + 1 - R) * ORA_B : 0;
        else elig_end = (size_t)s * ORA_B;
        if (elig_end > n) elig_end = n;
        if (elig_end > inserted) { global_insert(&e, inserted, elig_end); inserted = elig_end; }
        int64_t count = (int64_t)(s_end - s);
        int batch_rc = ORA_OK;
#ifdef _OPENMP
#pragma omp parallel for schedule(dynamic, 1) num_threads((int)e.p.threads)
#endif
        for (int64_t k = 0; k < count; k++) {
            int tid = 0;
#ifdef _OPENMP
            tid = omp_get_thread_num();
#endif
            uint64_t b = s + (uint64_t)k;
            uint32_t n_seq, n_lit;
            parse_block(&e, b, elig_end, &scr[tid], &n_seq, &n_lit, &blocks[b].st);
            int r2 = serialise_block(&e, b, &scr[tid], n_seq, n_lit, &blocks[b]);
            if (r2 != ORA_OK) {
#ifdef _OPENMP
#pragma omp critical
#endif
                batch_rc = r2;
            }
        }
        rc = batch_rc;
    }
    if (rc != ORA_OK) goto done;

    {   /* FORMAT.md section 1: header, index, payload */
        uint64_t index_bytes = (nb + 1) * 8 + nb * 3 * 32 * 4;
        uint64_t payload_off = pad16(ORA_HDR_BYTES + index_bytes);
        uint64_t payload = 0;
        for (uint64_t b = 0; b < nb; b++) payload += blocks[b].rec_bytes;
        if (payload_off + payload > cap) { rc = ORA_E_CAPACITY; goto done; }
        memset(out, 0, (size_t)payload_off);
        memcpy(out, "ACEAPEX1", 8);
        wr32(out + 8, 1);
        out[12] = ORA_BLOG; out[13] = (uint8_t)e.p.offset_width; out[14] = 32; out[15] = 12;
        wr64(out + 16, n); wr64(out + 24, nb);
        ora_enc_stats S;
        memset(&S, 0, sizeof S);
        uint8_t *rec_off = out + ORA_HDR_BYTES, *states = rec_off + (nb + 1) * 8;
        uint64_t o = 0;
        for (uint64_t b = 0; b < nb; b++) {
            wr64(rec_off + b * 8, o);
            memcpy(out + payload_off + o, blocks[b].rec, blocks[b].rec_bytes);
            o += blocks[b].rec_bytes;
            for (int k = 0; k < 3; k++)
                for (int l = 0; l < 32; l++) wr32(states + ((b * 3 + (uint64_t)k) * 32 + (uint64_t)l) * 4, blocks[b].states[k][l]);
            const ora_enc_stats *t = &blocks[b].st;
            S.n_seq += t->n_seq; S.n_lit += t->n_lit; S.match_bytes += t->match_bytes;
            S.intra_match_bytes += t->intra_match_bytes; S.n_extras += t->n_extras; S.table_bytes += t->table_bytes;
            for (int k = 0; k < 3; k++) { S.n_sym[k] += t->n_sym[k]; S.n_words[k] += t->n_words[k]; S.n_raw[k] += t->n_raw[k]; S.n_const[k] += t->n_const[k]; }
            if (t->max_depth_seen > S.max_depth_seen) S.max_depth_seen = t->max_depth_seen;
            if (t->max_level_seen > S.max_level_seen) S.max_level_seen = t->max_level_seen;
        }
        wr64(rec_off + nb * 8, o);
        wr32(out + 32, e.p.max_depth); wr32(out + 36, e.p.window);
        wr32(out + 40, S.max_level_seen); wr32(out + 44, e.p.min_match | e.p.max_fanout << 16);
        wr64(out + 48, ORA_HDR_BYTES); wr64(out + 56, payload_off);
        *out_len = (size_t)(payload_off + payload);
        if (stats) *stats = S;
    }
done:
    if (blocks) for (uint64_t b = 0; b < nb; b++) free(blocks[b].rec);
    if (scr) for (uint32_t t = 0; t < e.p.threads; t++) free(scr[t].fan_bits);
    free(blocks); free(scr); free(e.head); free(e.prev); free(e.depth); free(e.head2); free(e.prev2);
    return rc;
}
