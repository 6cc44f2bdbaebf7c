/* workloads/gen.c — seeded synthetic input generators (raw, uncompressed bytes only).
 *
 * This module serves BOTH the oracle and the CUDA path as the source of test/bench
 * inputs.  It holds none of the method's arithmetic: no LZ77, no offsets, no tokens,
 * no depth.  It only produces byte buffers whose statistics follow BASELINE.json's
 * five configs.  The paper's datasets (PAPER.md:81-87,
 * §4.2) are not reproduced; these buffers stand in for their shapes.
 *
 * PRNG: SplitMix64 (state += 0x9E3779B97F4A7C15; two xor-shift-multiply rounds).
 * Seed convention: 260604268 + config index (config 3 reuses config 1's seed).
 *
 * C ABI (all return 0 on success):
 *   wl_markov (out, n, seed)   config 0  order-2 Markov over 64 symbols + 20 % copied spans
 *   wl_text   (out, n, seed)   config 1/3 Zipf words, punctuation, XML-like tags, repeated lines
 *   wl_fastq  (out, n, seed)   config 2  4-line FASTQ-like records
 *   wl_stress (out, n, seed)   config 4  runs / random / text segments
 */
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#include <math.h>

typedef struct { uint64_t s; } rng_t;

static inline uint64_t rng_next(rng_t* r) {
    uint64_t z = (r->s += 0x9E3779B97F4A7C15ULL);
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
    return z ^ (z >> 31);
}
static inline double rng_u01(rng_t* r) { return (double)(rng_next(r) >> 11) * (1.0 / 9007199254740992.0); }
/* uniform integer in [0, n) */
static inline uint64_t rng_below(rng_t* r, uint64_t n) {
    return (uint64_t)(((unsigned __int128)rng_next(r) * n) >> 64);
}
/* uniform integer in [lo, hi] */
static inline uint64_t rng_range(rng_t* r, uint64_t lo, uint64_t hi) { return lo + rng_below(r, hi - lo + 1); }

/* ------------------------------------------------------------------ config 0 */
/* Order-2 Markov over 64 printable symbols; each of the 4096 contexts has a skewed
 * weight vector w_i = u_i^4.  Spans alternate: with probability 0.20 (and pos >= 4) a
 * copy span (length U[4,256], source uniform in [0,pos), byte-by-byte so it may
 * self-overlap), otherwise a Markov span of length U[4,256]. */
int wl_markov(uint8_t* out, uint64_t n, uint64_t seed) {
    rng_t r = { seed };
    static const char alpha[65] = "ABCDEFGHIJKLMNOPQRSTUVWXYZabcdefghijklmnopqrstuvwxyz0123456789 \n";
    float* cum = (float*)malloc(sizeof(float) * 4096 * 64);
    if (!cum) return -1;
    for (int c = 0; c < 4096; ++c) {
        double w[64], tot = 0;
        for (int i = 0; i < 64; ++i) { double u = rng_u01(&r); w[i] = u * u * u * u; tot += w[i]; }
        double acc = 0;
        for (int i = 0; i < 64; ++i) { acc += w[i] / tot; cum[c * 64 + i] = (float)acc; }
        cum[c * 64 + 63] = 2.0f;
    }
    uint64_t pos = 0; int a = 0, b = 0;
    while (pos < n) {
        uint64_t len = rng_range(&r, 4, 256);
        if (len > n - pos) len = n - pos;
        if (pos >= 4 && rng_u01(&r) < 0.20) {
            uint64_t src = rng_below(&r, pos);
            for (uint64_t i = 0; i < len; ++i) out[pos + i] = out[src + i];
            pos += len;
        } else {
            for (uint64_t i = 0; i < len; ++i) {
                float u = (float)rng_u01(&r);
                const float* cv = cum + ((a * 64 + b) << 6);
                int s = 0; while (cv[s] < u) ++s;
                out[pos + i] = (uint8_t)alpha[s];
                a = b; b = s;
            }
            pos += len;
        }
    }
    free(cum);
    return 0;
}

/* ------------------------------------------------------------------ config 1 / 3 */
#define VOCAB 50000
#define NTAGS 40
typedef struct {
    rng_t r;
    char   (*word)[16];     /* VOCAB words, NUL-free, length in wlen */
    uint8_t* wlen;
    double*  zcum;          /* Zipf(s=1.1) cumulative over ranks */
    char   tag[NTAGS][12]; uint8_t taglen[NTAGS];
    uint64_t* line_start;   /* absolute offsets of completed lines */
    uint32_t* line_len;
    uint64_t n_lines, cap_lines;
} text_t;

static int text_init(text_t* t, uint64_t seed) {
    memset(t, 0, sizeof *t);
    t->r.s = seed;
    t->word = malloc(sizeof(char[16]) * VOCAB);
    t->wlen = malloc(VOCAB);
    t->zcum = malloc(sizeof(double) * VOCAB);
    if (!t->word || !t->wlen || !t->zcum) return -1;
    /* seeded skewed letter distribution: weight 1/(k+4) over a seeded permutation */
    int perm[26]; for (int i = 0; i < 26; ++i) perm[i] = i;
    for (int i = 25; i > 0; --i) { int j = (int)rng_below(&t->r, (uint64_t)i + 1); int x = perm[i]; perm[i] = perm[j]; perm[j] = x; }
    double lc[26], acc = 0, tot = 0;
    for (int k = 0; k < 26; ++k) tot += 1.0 / (k + 4);
    for (int k = 0; k < 26; ++k) { acc += (1.0 / (k + 4)) / tot; lc[k] = acc; }
    lc[25] = 2.0;
    /* word length pmf over 1..14, peaked at 4-7; low ranks favour short words */
    static const double base[14] = { 2, 6, 10, 14, 14, 12, 10, 8, 6, 4, 3, 2, 1, 1 };
    for (int w = 0; w < VOCAB; ++w) {
        double pw[14], s = 0;
        for (int L = 0; L < 14; ++L) { pw[L] = base[L] * ((w < 200 && L < 4) ? 4.0 : 1.0); s += pw[L]; }
        double u = rng_u01(&t->r) * s, a2 = 0; int L = 0;
        for (; L < 13; ++L) { a2 += pw[L]; if (u < a2) break; }
        t->wlen[w] = (uint8_t)(L + 1);
        for (int i = 0; i <= L; ++i) {
            double v = rng_u01(&t->r); int k = 0; while (lc[k] < v) ++k;
            t->word[w][i] = (char)('a' + perm[k]);
        }
    }
    double z = 0;
    for (int w = 0; w < VOCAB; ++w) z += pow((double)(w + 1), -1.1);
    acc = 0;
    for (int w = 0; w < VOCAB; ++w) { acc += pow((double)(w + 1), -1.1) / z; t->zcum[w] = acc; }
    t->zcum[VOCAB - 1] = 2.0;
    for (int g = 0; g < NTAGS; ++g) {
        int L = (int)rng_range(&t->r, 3, 10);
        t->taglen[g] = (uint8_t)L;
        for (int i = 0; i < L; ++i) { double v = rng_u01(&t->r); int k = 0; while (lc[k] < v) ++k; t->tag[g][i] = (char)('a' + perm[k]); }
    }
    t->cap_lines = 1 << 16;
    t->line_start = malloc(sizeof(uint64_t) * t->cap_lines);
    t->line_len = malloc(sizeof(uint32_t) * t->cap_lines);
    return (t->line_start && t->line_len) ? 0 : -1;
}
static void text_free(text_t* t) { free(t->word); free(t->wlen); free(t->zcum); free(t->line_start); free(t->line_len); }

static inline int text_zipf(text_t* t) {
    double u = rng_u01(&t->r);
    int lo = 0, hi = VOCAB - 1;
    while (lo < hi) { int mid = (lo + hi) >> 1; if (t->zcum[mid] < u) lo = mid + 1; else hi = mid; }
    return lo;
}
#define PUT(c) do { if (pos < end) out[pos++] = (uint8_t)(c); } while (0)
/* Emit whole lines into out[pos, end); the last line is truncated at end.  Returns new pos. */
static uint64_t text_emit(text_t* t, uint8_t* out, uint64_t pos, uint64_t end) {
    static const char punct[6] = { ',', '.', ';', ':', '!', '?' };
    while (pos < end) {
        uint64_t ls = pos;
        if (t->n_lines > 0 && rng_u01(&t->r) < 0.15) {           /* verbatim copy of an earlier line */
            uint64_t k = rng_below(&t->r, t->n_lines);
            uint64_t s = t->line_start[k]; uint32_t L = t->line_len[k];
            for (uint32_t i = 0; i < L && pos < end; ++i) out[pos++] = out[s + i];
        } else {
            int tagged = rng_u01(&t->r) < 0.30, g = 0;
            if (tagged) {
                g = (int)rng_below(&t->r, NTAGS);
                PUT('<'); for (int i = 0; i < t->taglen[g]; ++i) PUT(t->tag[g][i]); PUT('>');
            }
            int done = 0;
            while (!done && pos < end) {
                int k = (int)rng_range(&t->r, 5, 20);
                for (int w = 0; w < k && pos < end; ++w) {
                    int id = text_zipf(t); int cap = rng_u01(&t->r) < 0.08;
                    for (int i = 0; i < t->wlen[id]; ++i) { char c = t->word[id][i]; if (cap && i == 0) c = (char)(c - 32); PUT(c); }
                    if (w + 1 < k) PUT(' ');
                }
                PUT(punct[rng_below(&t->r, 6)]);
                if (rng_u01(&t->r) < (1.0 / 3.0)) done = 1; else PUT(' ');
            }
            if (tagged) { PUT('<'); PUT('/'); for (int i = 0; i < t->taglen[g]; ++i) PUT(t->tag[g][i]); PUT('>'); }
            PUT('\n');
        }
        if (t->n_lines == t->cap_lines) {
            t->cap_lines *= 2;
            t->line_start = realloc(t->line_start, sizeof(uint64_t) * t->cap_lines);
            t->line_len = realloc(t->line_len, sizeof(uint32_t) * t->cap_lines);
            if (!t->line_start || !t->line_len) return end;
        }
        t->line_start[t->n_lines] = ls; t->line_len[t->n_lines] = (uint32_t)(pos - ls); t->n_lines++;
    }
    return pos;
}

int wl_text(uint8_t* out, uint64_t n, uint64_t seed) {
    text_t t; if (text_init(&t, seed)) return -1;
    text_emit(&t, out, 0, n);
    text_free(&t);
    return 0;
}

/* ------------------------------------------------------------------ config 2 */
static inline uint64_t put_uint(uint8_t* out, uint64_t pos, uint64_t end, uint64_t v) {
    char buf[24]; int k = 0;
    do { buf[k++] = (char)('0' + v % 10); v /= 10; } while (v);
    while (k-- > 0) PUT(buf[k]);
    return pos;
}
int wl_fastq(uint8_t* out, uint64_t n, uint64_t seed) {
    rng_t r = { seed };
    const uint64_t REF = 5000000; const int RL = 150;
    uint8_t* ref = malloc(REF); if (!ref) return -1;
    static const char acgt[4] = { 'A', 'C', 'G', 'T' };
    for (uint64_t i = 0; i < REF; ++i) ref[i] = (uint8_t)acgt[rng_next(&r) >> 62];
    /* step pmf over {-3..+2}: mid-read mean ~ 0, first/last 20 positions mean ~ -0.5 */
    static const double pm[6] = { 0.03, 0.07, 0.20, 0.40, 0.20, 0.10 };
    static const double pe[6] = { 0.08, 0.14, 0.28, 0.30, 0.14, 0.06 };
    uint64_t pos = 0, end = n, rec = 0;
    uint64_t lane = 1, tile = 1101, x = 1000, y = 1000;
    while (pos < end) {
        /* header */
        const char* h = "@SIM:001:"; for (int i = 0; h[i]; ++i) PUT(h[i]);
        pos = put_uint(out, pos, end, lane); PUT(':');
        pos = put_uint(out, pos, end, tile); PUT(':');
        pos = put_uint(out, pos, end, x);    PUT(':');
        pos = put_uint(out, pos, end, y);    PUT('\n');
        x += rng_range(&r, 1, 60);
        if (x > 20000) { x = 1000 + rng_below(&r, 100); y += rng_range(&r, 1, 40); }
        if (y > 20000) { y = 1000 + rng_below(&r, 100); tile += 1; }
        if (tile > 2228) tile = 1101;
        if (++rec % 400000 == 0) lane = lane % 8 + 1;
        /* read */
        uint64_t s = rng_below(&r, REF - RL);
        for (int i = 0; i < RL; ++i) {
            uint8_t c = ref[s + i];
            double u = rng_u01(&r);
            if (u < 0.001) c = 'N';
            else if (u < 0.011) c = (uint8_t)acgt[rng_next(&r) >> 62];
            PUT(c);
        }
        PUT('\n'); PUT('+'); PUT('\n');
        /* quality */
        int q = (int)rng_range(&r, 30, 40);
        for (int i = 0; i < RL; ++i) {
            PUT(q + 33);
            const double* p = (i < 20 || i >= RL - 20) ? pe : pm;
            double u = rng_u01(&r), a = 0; int k = 0;
            for (; k < 5; ++k) { a += p[k]; if (u < a) break; }
            q += k - 3; if (q < 2) q = 2; if (q > 41) q = 41;
        }
        PUT('\n');
    }
    free(ref);
    return 0;
}

/* ------------------------------------------------------------------ config 4 */
int wl_stress(uint8_t* out, uint64_t n, uint64_t seed) {
    rng_t r = { seed };
    text_t t; if (text_init(&t, seed ^ 0x5EEDULL)) return -1;
    uint64_t pos = 0;
    while (pos < n) {
        uint64_t seg = rng_range(&r, 64 * 1024, 4 * 1024 * 1024);
        uint64_t end = pos + seg < n ? pos + seg : n;
        double u = rng_u01(&r);
        if (u < 0.4) {                                   /* runs: period 1 (p=0.5) or U[2,16] */
            while (pos < end) {
                int period = rng_u01(&r) < 0.5 ? 1 : (int)rng_range(&r, 2, 16);
                uint8_t pat[16]; for (int i = 0; i < period; ++i) pat[i] = (uint8_t)(rng_next(&r) >> 56);
                double lg = log(32.0) + rng_u01(&r) * (log(262144.0) - log(32.0));
                uint64_t L = (uint64_t)exp(lg);
                for (uint64_t i = 0; i < L && pos < end; ++i) out[pos++] = pat[i % (uint64_t)period];
            }
        } else if (u < 0.7) {                            /* incompressible */
            while (pos + 8 <= end) { uint64_t v = rng_next(&r); memcpy(out + pos, &v, 8); pos += 8; }
            while (pos < end) out[pos++] = (uint8_t)(rng_next(&r) >> 56);
        } else {                                         /* text, generator state carried across segments */
            pos = text_emit(&t, out, pos, end);
        }
    }
    text_free(&t);
    return 0;
}
