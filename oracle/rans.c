/* ORACLE (test infrastructure) — entropy layer: FORMAT.md section 3, PAPER.md:33 (per-block ANS),
 * PAPER.md:124 ref [6] (interleaved rANS). Written in the order and notation of FORMAT.md. */
#include "aceapex_oracle.h"

#include <stdlib.h>
#include <string.h>

#define PROB_BITS 12u
#define M_TOTAL 4096u  /* 2^PROB_BITS */
#define RANS_L 65536u  /* lower bound of the state interval [2^16, 2^32) */

/* FORMAT.md section 3 "Quantiser". */
void ora_quantise(const uint32_t count[256], uint16_t freq[256])
{
    uint64_t n = 0;
    int order[256], n_present = 0;
    int64_t sum = 0;
    for (int s = 0; s < 256; s++) n += count[s];
    memset(freq, 0, 256 * sizeof(uint16_t));
    if (n == 0) return;
    for (int s = 0; s < 256; s++) {
        if (!count[s]) continue;
        uint64_t f = ((uint64_t)count[s] * M_TOTAL) / n;
        if (f < 1) f = 1;
        freq[s] = (uint16_t)f;
        sum += (int64_t)f;
        order[n_present++] = s;
    }
    /* order of decreasing count, ties to the lower symbol value (insertion sort, <= 256 items) */
    for (int i = 1; i < n_present; i++) {
        int s = order[i], j = i - 1;
        while (j >= 0 && count[order[j]] < count[s]) { order[j + 1] = order[j]; j--; }
        order[j + 1] = s;
    }
    int64_t diff = (int64_t)M_TOTAL - sum;
    if (diff > 0) {
        freq[order[0]] = (uint16_t)(freq[order[0]] + diff);
    } else {
        for (int i = 0; i < n_present && diff < 0; i++) {
            int s = order[i];
            int64_t take = (int64_t)freq[s] - 1;
            if (take > -diff) take = -diff;
            freq[s] = (uint16_t)(freq[s] - take);
            diff += take;
        }
    }
}

static int cumulative(const uint16_t freq[256], uint32_t cum[257])
{
    uint32_t c = 0;
    for (int s = 0; s < 256; s++) { cum[s] = c; c += freq[s]; }
    cum[256] = c;
    return c == M_TOTAL ? ORA_OK : ORA_E_ARG;
}

/* FORMAT.md section 3 "Encoder". */
int ora_rans_encode(const uint8_t *sym, size_t n, const uint16_t freq[256], uint32_t lanes,
                    uint32_t *states_out, uint16_t *words_out, size_t *n_words_out)
{
    uint32_t cum[257], x[32];
    size_t nw = 0;
    if (lanes < 1 || lanes > 32) return ORA_E_ARG;
    for (uint32_t l = 0; l < lanes; l++) x[l] = RANS_L;
    if (n == 0) {
        for (uint32_t l = 0; l < lanes; l++) states_out[l] = x[l];
        *n_words_out = 0;
        return ORA_OK;
    }
    if (cumulative(freq, cum) != ORA_OK) return ORA_E_ARG;
    for (size_t i = n; i-- > 0;) {
        uint32_t l = (uint32_t)(i % lanes);
        uint32_t f = freq[sym[i]], c = cum[sym[i]];
        if (f == 0) return ORA_E_ARG;
        if ((uint64_t)x[l] >= ((uint64_t)f << 20)) {
            words_out[nw++] = (uint16_t)(x[l] & 0xFFFFu);
            x[l] >>= 16;
        }
        x[l] = ((x[l] / f) << PROB_BITS) + (x[l] % f) + c;
    }
    for (size_t a = 0, b = nw; a + 1 < b; a++, b--) { /* reverse: decoder reads forward */
        uint16_t t = words_out[a]; words_out[a] = words_out[b - 1]; words_out[b - 1] = t;
    }
    for (uint32_t l = 0; l < lanes; l++) states_out[l] = x[l];
    *n_words_out = nw;
    return ORA_OK;
}

/* FORMAT.md section 3 "Decoder" (sequential semantics). */
int ora_rans_decode(const uint32_t *states, uint32_t lanes, const uint16_t *words, size_t n_words,
                    const uint16_t freq[256], uint8_t *sym_out, size_t n)
{
    uint32_t cum[257], x[32];
    uint8_t slot2sym[M_TOTAL];
    size_t w = 0;
    if (lanes < 1 || lanes > 32) return ORA_E_ARG;
    for (uint32_t l = 0; l < lanes; l++) x[l] = states[l];
    if (n > 0) {
        if (cumulative(freq, cum) != ORA_OK) return ORA_E_CORRUPT;
        for (int s = 0; s < 256; s++)
            for (uint32_t k = cum[s]; k < cum[s + 1]; k++) slot2sym[k] = (uint8_t)s;
    }
    for (size_t i = 0; i < n; i++) {
        uint32_t l = (uint32_t)(i % lanes);
        uint32_t slot = x[l] & (M_TOTAL - 1);
        uint32_t s = slot2sym[slot];
        x[l] = freq[s] * (x[l] >> PROB_BITS) + slot - cum[s];
        if (x[l] < RANS_L) {
            if (w >= n_words) return ORA_E_CORRUPT;
            x[l] = (x[l] << 16) | words[w++];
        }
        sym_out[i] = (uint8_t)s;
    }
    if (w != n_words) return ORA_E_CORRUPT;
    for (uint32_t l = 0; l < lanes; l++)
        if (x[l] != RANS_L) return ORA_E_CORRUPT;
    return ORA_OK;
}

/* FNV-1a, 64-bit: offset basis 0xcbf29ce484222325, prime 0x100000001b3. */
uint64_t ora_fnv1a64(const void *data, size_t n)
{
    const uint8_t *p = (const uint8_t *)data;
    uint64_t h = 0xcbf29ce484222325ull;
    for (size_t i = 0; i < n; i++) { h ^= p[i]; h *= 0x100000001b3ull; }
    return h;
}

const char *ora_strerror(int code)
{
    switch (code) {
    case ORA_OK: return "ok";
    case ORA_E_ARG: return "bad argument";
    case ORA_E_FORMAT: return "bad header";
    case ORA_E_CAPACITY: return "output capacity too small";
    case ORA_E_CORRUPT: return "corrupt container";
    case ORA_E_RANGE: return "out of range";
    case ORA_E_NOMEM: return "out of memory";
    case ORA_E_PROMISE: return "header promise violated";
    default: return "unknown";
    }
}
