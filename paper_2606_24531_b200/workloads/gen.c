/*
 * Seeded synthetic workload generators (BASELINE.json configs[0..4]; recipe in DESIGN.md).
 *
 * These stand in for the paper's datasets (real FASTQ NA12878, a repetitive genome, enwik9,
 * silesia: PAPER.md:65-68), none of which is available. The module holds no codec arithmetic:
 * it only writes bytes. Both the oracle (tests, bench) and the CUDA path consume its output.
 *
 * Randomness: splitmix64 counter mixer; Gaussian = sum of 12 uniforms - 6; libm is used only
 * for the Zipf table (pow) and the geometric segment length (log).
 */
#include <math.h>
#include <stddef.h>
#include <stdint.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

typedef struct { uint64_t s; } rng_t;

static inline uint64_t rng_next(rng_t *r)
{
    uint64_t z = (r->s += 0x9E3779B97F4A7C15ull);
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
    return z ^ (z >> 31);
}
static inline uint32_t rng_below(rng_t *r, uint32_t n) { return (uint32_t)(((rng_next(r) >> 32) * (uint64_t)n) >> 32); }
static inline double rng_uniform(rng_t *r) { return (double)(rng_next(r) >> 11) * (1.0 / 9007199254740992.0); }
static inline double rng_gauss(rng_t *r)
{
    double s = 0;
    for (int i = 0; i < 12; i++) s += rng_uniform(r);
    return s - 6.0;
}

/* A generator is a producer of "units" (a record, a segment piece, a sentence) into a pending
 * buffer that fill() drains, so that a generator can be resumed across chunks (config 5). */
typedef struct gen gen_t;
struct gen {
    int kind;
    rng_t rng;
    uint8_t *pend;
    size_t pend_len, pend_pos, pend_cap;
    /* markov */
    uint8_t *succ; uint8_t *nsucc; int a, b;
    /* fastq */
    uint64_t read_id;
    /* genome */
    uint8_t *base; size_t base_len; size_t seg_pos, seg_left;
    /* text */
    char *vocab; uint32_t *voff; uint8_t *vlen; double *cdf; uint32_t n_vocab; int col;
};

enum { K_MARKOV = 0, K_FASTQ = 1, K_GENOME = 2, K_TEXT = 3, K_RANDOM = 4, K_MIXED = 5 };

static void pend_reserve(gen_t *g, size_t n)
{
    if (g->pend_cap < n) { g->pend = (uint8_t *)realloc(g->pend, n); g->pend_cap = n; }
}

/* ---- config 0: order-2 Markov text over 64 ASCII symbols -------------------------------- */
static const char MARKOV_ALPHA[] = "abcdefghijklmnopqrstuvwxyzABCDEFGHIJKLMNOPQRSTUVWXYZ .,;:!?'-()\n\"";
#define MARKOV_A 64

static void markov_init(gen_t *g)
{
    g->succ = (uint8_t *)malloc(MARKOV_A * MARKOV_A * 8);
    g->nsucc = (uint8_t *)malloc(MARKOV_A * MARKOV_A);
    for (int c = 0; c < MARKOV_A * MARKOV_A; c++) {
        g->nsucc[c] = (uint8_t)(2 + rng_below(&g->rng, 6));               /* 2..7 successors */
        for (int j = 0; j < 8; j++) g->succ[c * 8 + j] = (uint8_t)rng_below(&g->rng, MARKOV_A);
    }
    g->a = 0; g->b = 1;
}
static void markov_unit(gen_t *g)
{
    pend_reserve(g, 4096);
    for (int i = 0; i < 4096; i++) {
        int c = g->a * MARKOV_A + g->b, j = 0;
        while (j < g->nsucc[c] - 1 && (rng_next(&g->rng) & 1)) j++;       /* geometric weights */
        int s = g->succ[c * 8 + j];
        g->pend[i] = (uint8_t)MARKOV_ALPHA[s];
        g->a = g->b; g->b = s;
    }
    g->pend_len = 4096;
}

/* ---- config 1: FASTQ records -------------------------------------------------------------- */
static void fastq_unit(gen_t *g)
{
    pend_reserve(g, 512);
    int m = snprintf((char *)g->pend, 64, "@SYN.%llu\n", (unsigned long long)g->read_id++);
    uint8_t *p = g->pend + m;
    for (int i = 0; i < 150; i++)
        *p++ = (rng_below(&g->rng, 1000) == 0) ? 'N' : (uint8_t)"ACGT"[rng_below(&g->rng, 4)]; /* 0.1% N */
    *p++ = '\n'; *p++ = '+'; *p++ = '\n';
    for (int i = 0; i < 150; i++) {
        double mu = 38.0 - 13.0 * (double)i / 149.0;                      /* mean 38 -> 25 */
        double v = mu + 4.0 * rng_gauss(&g->rng);                         /* sd 4 */
        int q = (int)(v + 0.5);
        if (q < 2) q = 2;
        if (q > 41) q = 41;
        *p++ = (uint8_t)(33 + q);                                         /* Phred+33 */
    }
    *p++ = '\n';
    g->pend_len = (size_t)(p - g->pend);
}

/* ---- config 2: repetitive genome ---------------------------------------------------------- */
static void genome_init(gen_t *g)
{
    g->base_len = 2000000;
    g->base = (uint8_t *)malloc(g->base_len);
    for (size_t i = 0; i < g->base_len; i++) g->base[i] = (uint8_t)"ACGT"[rng_below(&g->rng, 4)];
    g->seg_left = 0;
}
static void genome_unit(gen_t *g)
{
    pend_reserve(g, 4096);
    size_t k = 0;
    while (k < 4096) {
        if (g->seg_left == 0) {
            /* geometric length, mean ~10 kbp, clipped to [1, 50] kbp */
            double u = rng_uniform(&g->rng);
            size_t len = (size_t)(-log(1.0 - u) * 10000.0);
            if (len < 1000) len = 1000;
            if (len > 50000) len = 50000;
            g->seg_pos = rng_below(&g->rng, (uint32_t)(g->base_len - len));
            g->seg_left = len;
        }
        uint8_t c = g->base[g->seg_pos++];
        g->seg_left--;
        if (rng_below(&g->rng, 100) == 0) {                               /* 1% point substitutions */
            uint8_t d;
            do d = (uint8_t)"ACGT"[rng_below(&g->rng, 4)]; while (d == c);
            c = d;
        }
        g->pend[k++] = c;
    }
    g->pend_len = k;
}

/* ---- config 3: English-like text ---------------------------------------------------------- */
static void text_init(gen_t *g)
{
    static const char LETTERS[] =
        "eeeeeeeeeeeetttttttttaaaaaaaaoooooooiiiiiiinnnnnnnsssssshhhhhhrrrrrrddddllllcccuuummmwwffggyyppbbvkjxqz";
    const uint32_t nl = (uint32_t)(sizeof LETTERS - 1);
    g->n_vocab = 50000;
    g->vocab = (char *)malloc((size_t)g->n_vocab * 12);
    g->voff = (uint32_t *)malloc(sizeof(uint32_t) * g->n_vocab);
    g->vlen = (uint8_t *)malloc(g->n_vocab);
    g->cdf = (double *)malloc(sizeof(double) * g->n_vocab);
    uint32_t o = 0;
    for (uint32_t w = 0; w < g->n_vocab; w++) {
        uint32_t len = 2 + rng_below(&g->rng, 11);                        /* 2..12 letters */
        g->voff[w] = o; g->vlen[w] = (uint8_t)len;
        for (uint32_t i = 0; i < len; i++) g->vocab[o++] = LETTERS[rng_below(&g->rng, nl)];
    }
    double s = 0;
    for (uint32_t w = 0; w < g->n_vocab; w++) { s += 1.0 / pow((double)w + 1.0, 1.1); g->cdf[w] = s; } /* Zipf s=1.1 */
    for (uint32_t w = 0; w < g->n_vocab; w++) g->cdf[w] /= s;
    g->col = 0;
}
static void text_unit(gen_t *g)
{
    pend_reserve(g, 26 * 14 + 16);
    uint32_t nw = 8 + rng_below(&g->rng, 18);                             /* sentence of 8..25 words */
    size_t k = 0;
    for (uint32_t i = 0; i < nw; i++) {
        double u = rng_uniform(&g->rng);
        uint32_t lo = 0, hi = g->n_vocab - 1;
        while (lo < hi) { uint32_t mid = (lo + hi) / 2; if (g->cdf[mid] < u) lo = mid + 1; else hi = mid; }
        memcpy(g->pend + k, g->vocab + g->voff[lo], g->vlen[lo]);
        k += g->vlen[lo];
        if (i == nw - 1) g->pend[k++] = '.';
        g->col += g->vlen[lo] + 1;
        if (g->col >= 80) { g->pend[k++] = '\n'; g->col = 0; } else g->pend[k++] = ' ';
    }
    g->pend_len = k;
}

/* ---- uniform random bytes ----------------------------------------------------------------- */
static void random_unit(gen_t *g)
{
    pend_reserve(g, 4096);
    for (int i = 0; i < 4096; i += 8) { uint64_t v = rng_next(&g->rng); memcpy(g->pend + i, &v, 8); }
    g->pend_len = 4096;
}

static gen_t *gen_new(int kind, uint64_t seed)
{
    gen_t *g = (gen_t *)calloc(1, sizeof *g);
    g->kind = kind;
    g->rng.s = seed;
    g->read_id = 1;
    if (kind == K_MARKOV) markov_init(g);
    else if (kind == K_GENOME) genome_init(g);
    else if (kind == K_TEXT) text_init(g);
    return g;
}
static void gen_free(gen_t *g)
{
    if (!g) return;
    free(g->pend); free(g->succ); free(g->nsucc); free(g->base);
    free(g->vocab); free(g->voff); free(g->vlen); free(g->cdf); free(g);
}
static void gen_fill(gen_t *g, uint8_t *out, size_t n)
{
    size_t k = 0;
    while (k < n) {
        if (g->pend_pos >= g->pend_len) {
            g->pend_pos = 0;
            switch (g->kind) {
            case K_MARKOV: markov_unit(g); break;
            case K_FASTQ: fastq_unit(g); break;
            case K_GENOME: genome_unit(g); break;
            case K_TEXT: text_unit(g); break;
            default: random_unit(g); break;
            }
        }
        size_t take = g->pend_len - g->pend_pos;
        if (take > n - k) take = n - k;
        memcpy(out + k, g->pend + g->pend_pos, take);
        g->pend_pos += take; k += take;
    }
}

/* kind: 0 markov, 1 fastq, 2 genome, 3 text, 4 random, 5 mixed (64 KiB chunks, exactly 25% each of
 * fastq / genome / text / random in a seeded order; each generator continues across its chunks).
 * Returns 0, or -1 on a bad kind. */
int aceapex_workload_generate(int kind, uint64_t seed, uint8_t *out, size_t n)
{
    if (kind < 0 || kind > K_MIXED || (!out && n)) return -1;
    if (kind != K_MIXED) {
        gen_t *g = gen_new(kind, seed);
        gen_fill(g, out, n);
        gen_free(g);
        return 0;
    }
    const size_t chunk = 65536;
    const size_t n_chunks = (n + chunk - 1) / chunk;
    uint8_t *order = (uint8_t *)malloc(n_chunks ? n_chunks : 1);
    for (size_t i = 0; i < n_chunks; i++) order[i] = (uint8_t)(i & 3);     /* exactly 25% each */
    rng_t sh = { seed + 0x60 };
    for (size_t i = n_chunks; i > 1; i--) {                                /* Fisher-Yates */
        size_t j = (size_t)(rng_next(&sh) % i);
        uint8_t t = order[i - 1]; order[i - 1] = order[j]; order[j] = t;
    }
    gen_t *sub[4] = { gen_new(K_FASTQ, seed + 0x10), gen_new(K_GENOME, seed + 0x20),
                      gen_new(K_TEXT, seed + 0x30), gen_new(K_RANDOM, seed + 0x40) };
    for (size_t c = 0; c < n_chunks; c++) {
        size_t off = c * chunk, len = (n - off < chunk) ? n - off : chunk;
        gen_fill(sub[order[c]], out + off, len);
    }
    for (int i = 0; i < 4; i++) gen_free(sub[i]);
    free(order);
    return 0;
}
