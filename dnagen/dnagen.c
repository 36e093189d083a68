/*
 * dnagen.c -- seeded synthetic DNA input generators (inputs only).
 *
 * This file holds NO tokenizer arithmetic: it produces the byte buffers, record
 * offsets and merge tables that stand in for the paper's workloads (synthetic
 * equal-length strings) in the five BASELINE.json
 * configs.  Both the CPU oracle's tests and the CUDA path's tests/bench read the
 * same generated inputs; neither the oracle nor the CUDA library links this file.
 *
 * Determinism: every record is drawn from its own xoshiro256** stream seeded by
 * splitmix64 over (seed, config, record index), so output does not depend on how
 * the caller splits records across threads.  No libc rand(), no libm
 * distributions: results are identical on every box.
 */
#include <stdint.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

typedef struct { uint64_t s[4]; } rng_t;

static uint64_t splitmix64(uint64_t *x) {
    uint64_t z = (*x += 0x9E3779B97F4A7C15ULL);
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
    return z ^ (z >> 31);
}

static void rng_seed(rng_t *r, uint64_t seed, uint64_t a, uint64_t b) {
    uint64_t x = seed ^ (a * 0xD1B54A32D192ED03ULL) ^ (b * 0x8CB92BA72F3D8DD7ULL);
    for (int i = 0; i < 4; ++i) r->s[i] = splitmix64(&x);
}

static inline uint64_t rotl(uint64_t x, int k) { return (x << k) | (x >> (64 - k)); }

static inline uint64_t rng_next(rng_t *r) {
    uint64_t *s = r->s;
    uint64_t result = rotl(s[1] * 5, 7) * 9, t = s[1] << 17;
    s[2] ^= s[0]; s[3] ^= s[1]; s[1] ^= s[2]; s[0] ^= s[3];
    s[2] ^= t; s[3] = rotl(s[3], 45);
    return result;
}

/* uniform double in [0,1) with 53 bits */
static inline double rng_u01(rng_t *r) { return (double)(rng_next(r) >> 11) * (1.0 / 9007199254740992.0); }

/* uniform integer in [0, n) (n > 0); multiply-shift, bias < 2^-32 for n < 2^32 */
static inline uint64_t rng_below(rng_t *r, uint64_t n) {
    return (uint64_t)(((__uint128_t)rng_next(r) * n) >> 64);
}

static const char ACGT[4] = {'A', 'C', 'G', 'T'};

/* ------------------------------------------------------------------------- */
/* Order-2 Markov table (configs 2 and 4).  64 doubles: for context (b[i-2],
 * b[i-1]) = ctx in 0..15, cumulative probabilities of A,C,G,T.  Base rates
 * (A .295, C .205, G .205, T .295) give GC 0.41; each context perturbs them by a
 * factor in [0.8, 1.2] and renormalises.                                     */
void dnagen_markov_table(uint64_t seed, double *cum /* [16][4] */) {
    static const double base[4] = {0.295, 0.205, 0.205, 0.295};
    rng_t r; rng_seed(&r, seed, 0x4D41524BULL /* 'MARK' */, 0);
    for (int c = 0; c < 16; ++c) {
        double p[4], tot = 0.0;
        for (int j = 0; j < 4; ++j) { p[j] = base[j] * (0.8 + 0.4 * rng_u01(&r)); tot += p[j]; }
        double acc = 0.0;
        for (int j = 0; j < 4; ++j) { acc += p[j] / tot; cum[c * 4 + j] = acc; }
        cum[c * 4 + 3] = 1.0;
    }
}

/* ------------------------------------------------------------------------- */
/* One record.  model: 0 = i.i.d. uniform ACGT, 1 = order-2 Markov (cum != NULL).
 * p_n: each base independently replaced by 'N'.  p_lower: each base byte
 * independently lower-cased (N included).  header != 0: write
 * ">r<rec> len=<n_bases>\n" first.  line_width > 0: '\n' after every line_width
 * bases and after a final partial line.  term_newline != 0 (only with
 * line_width == 0): one '\n' after the last base.
 * Returns bytes written.  dst == NULL: only count.                            */
int64_t dnagen_record(uint8_t *dst, int64_t n_bases, uint64_t seed, uint64_t cfg, uint64_t rec,
                      int model, const double *cum, double p_n, double p_lower,
                      int header, int line_width, int term_newline) {
    int64_t w = 0;
    if (header) {
        char buf[64];
        int h = snprintf(buf, sizeof buf, ">r%llu len=%lld\n", (unsigned long long)rec, (long long)n_bases);
        if (dst) memcpy(dst, buf, (size_t)h);
        w += h;
    }
    if (!dst) {
        w += n_bases;
        if (line_width > 0) w += (n_bases + line_width - 1) / line_width;
        else if (term_newline) w += 1;
        return w;
    }
    rng_t r; rng_seed(&r, seed, cfg, rec);
    int c1 = (int)rng_below(&r, 4), c2 = (int)rng_below(&r, 4);  /* Markov warm-up context */
    for (int64_t i = 0; i < n_bases; ++i) {
        int b;
        if (model == 1) {
            const double *row = cum + (c1 * 4 + c2) * 4;
            double u = rng_u01(&r);
            b = (u < row[0]) ? 0 : (u < row[1]) ? 1 : (u < row[2]) ? 2 : 3;
            c1 = c2; c2 = b;
        } else {
            b = (int)(rng_next(&r) >> 62);
        }
        uint8_t ch = (uint8_t)ACGT[b];
        if (p_n > 0.0 && rng_u01(&r) < p_n) ch = 'N';
        if (p_lower > 0.0 && rng_u01(&r) < p_lower) ch |= 0x20;
        dst[w++] = ch;
        if (line_width > 0 && (i + 1) % line_width == 0) dst[w++] = '\n';
    }
    if (line_width > 0) { if (n_bases % line_width != 0) dst[w++] = '\n'; }
    else if (term_newline) dst[w++] = '\n';
    return w;
}

/* Fill records [r0, r1) of a flat buffer; offsets[r] is record r's first byte. */
void dnagen_fill_records(uint8_t *flat, const int64_t *offsets, const int64_t *n_bases, int64_t r0, int64_t r1,
                         uint64_t seed, uint64_t cfg, int model, const double *cum, double p_n, double p_lower,
                         int header, int line_width, int term_newline) {
    for (int64_t r = r0; r < r1; ++r)
        dnagen_record(flat + offsets[r], n_bases[r], seed, cfg, (uint64_t)r, model, cum, p_n, p_lower,
                      header, line_width, term_newline);
}

/* ------------------------------------------------------------------------- */
/* Config 2: runs of 'N', lengths uniform 1..max_len, starts uniform over the
 * flat base array, until frac of the bytes are N.  Runs may cross records.    */
int64_t dnagen_n_runs(uint8_t *flat, int64_t n, uint64_t seed, double frac, int max_len) {
    rng_t r; rng_seed(&r, seed, 0x4E52554EULL /* 'NRUN' */, 0);
    int64_t target = (int64_t)(frac * (double)n), covered = 0, runs = 0;
    while (covered < target) {
        int64_t len = 1 + (int64_t)rng_below(&r, (uint64_t)max_len);
        int64_t st = (int64_t)rng_below(&r, (uint64_t)n);
        for (int64_t i = st; i < st + len && i < n; ++i)
            if (flat[i] != 'N') { flat[i] = 'N'; ++covered; }
        ++runs;
    }
    return runs;
}

/* ------------------------------------------------------------------------- */
/* Record lengths.                                                             */
void dnagen_lengths_uniform(int64_t *out, int64_t n, int64_t lo, int64_t hi, uint64_t seed, uint64_t cfg) {
    rng_t r; rng_seed(&r, seed, cfg, 0x4C454EULL /* 'LEN' */);
    for (int64_t i = 0; i < n; ++i) out[i] = lo + (int64_t)rng_below(&r, (uint64_t)(hi - lo + 1));
}

/* log-uniform in [lo, hi] without libm: length = lo * 2^(u*log2(hi/lo)) is
 * evaluated as an integer power-of-two octave plus a linear mantissa, which is
 * log-uniform across octaves and uniform inside one (exact for the statistics
 * the tests pin: range and median).  Draw until total_bases is reached; the last
 * length is truncated.  Returns the number of records (<= max_n).            */
int64_t dnagen_lengths_loguniform(int64_t *out, int64_t max_n, int64_t total_bases, int64_t lo, int64_t hi,
                                  uint64_t seed, uint64_t cfg) {
    rng_t r; rng_seed(&r, seed, cfg, 0x4C4F47ULL /* 'LOG' */);
    int octaves = 0; while ((lo << (octaves + 1)) <= hi) ++octaves;   /* hi >= lo * 2^octaves */
    int64_t n = 0, tot = 0;
    while (tot < total_bases && n < max_n) {
        int64_t len;
        do {
            int o = (int)rng_below(&r, (uint64_t)(octaves + 1));
            int64_t base = lo << o;
            len = base + (int64_t)rng_below(&r, (uint64_t)base);
        } while (len > hi);
        if (tot + len > total_bases) len = total_bases - tot;
        out[n++] = len; tot += len;
    }
    return n;
}

/* ------------------------------------------------------------------------- */
/* Config 4 merge table ("simulated pair frequency"): draw a
 * corpus of corpus_bases from the Markov chain (no N); at each of n_merges
 * steps pick one adjacent position uniformly at random -- its pair is thereby
 * chosen with probability proportional to that pair's adjacent-occurrence count
 * -- record (left, right) as rule `step` with product token 4 + step, and
 * replace every occurrence left to right.  Rules are unique and refer only to
 * earlier tokens by construction.  Returns the number of rules written (stops
 * early if the corpus shrinks to one token).  This trains an INPUT; it is not
 * the encoder under test and shares nothing with it.                         */
int dnagen_merge_table(int32_t *merges /* [n_merges][2] */, int n_merges, int64_t corpus_bases,
                       uint64_t seed, const double *cum) {
    int32_t *tok = (int32_t *)malloc((size_t)corpus_bases * sizeof(int32_t));
    if (!tok) return -1;
    rng_t r; rng_seed(&r, seed, 0x434F5250ULL /* 'CORP' */, 0);
    int c1 = (int)rng_below(&r, 4), c2 = (int)rng_below(&r, 4);
    for (int64_t i = 0; i < corpus_bases; ++i) {
        const double *row = cum + (c1 * 4 + c2) * 4;
        double u = rng_u01(&r);
        int b = (u < row[0]) ? 0 : (u < row[1]) ? 1 : (u < row[2]) ? 2 : 3;
        c1 = c2; c2 = b; tok[i] = b;
    }
    int64_t n = corpus_bases;
    int step = 0;
    for (; step < n_merges && n >= 2; ++step) {
        int64_t j = (int64_t)rng_below(&r, (uint64_t)(n - 1));
        int32_t L = tok[j], R = tok[j + 1], P = 4 + step;
        merges[2 * step] = L; merges[2 * step + 1] = R;
        int64_t w = 0;
        for (int64_t i = 0; i < n;) {
            if (i + 1 < n && tok[i] == L && tok[i + 1] == R) { tok[w++] = P; i += 2; }
            else tok[w++] = tok[i++];
        }
        n = w;
    }
    free(tok);
    return step;
}
