/*
 * dnatok_oracle.c -- plain, slow, obviously-correct CPU definition of what the
 * DNATok hot path computes.  TEST INFRASTRUCTURE ONLY.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
 * reference legs may build, load or call this file.  The product (CUDA) path
 * shares no code, header, table or helper with it and never routes through it.
 *
 * The result is a deterministic integer function with exactly one correct answer
 * per input, so the oracle is the definition written out as the slowest obvious
 * loops, one record at a time, one byte at a time, in the order of SURVEY.md
 * section 8(c) steps 1-6.  Sources:
 *   - 256-entry ASCII->ID look-up table, case-insensitive A/C/G/T, N:
 *     (section 2.2, bytes path), PAPER.md:88 (Algorithm 1, l.8-16 and l.24-37).
 *   - non-overlapping k-mers, "length k, stride k":  PAPER.md:88 (Alg. 1 l.18),
 *     PAPER.md:115-117 (Alg. 2 l.7-8, MapKmer).
 *   - left padding "right-aligning the original T positions":
 *     (Alg. 2 l.12-14).
 *   - everything the paper is silent on (newline/header stripping, base-4 closed
 *     form, N-window -> UNK, tail policy, BPE lowest-rank-first merges, CSR
 *     offsets, attention mask):  BASELINE.json north_star, with the readings
 *     Q1-Q17 of SURVEY.md section 8(c), restated in DESIGN.md.
 *
 * Pins (tests/test_oracle_*.py, none of which re-type these loops): the paper's
 * self-test string ACGTNacgtn, the hand-worked example of SURVEY.md
 * section 8(c), closed forms (Q7 worked values, numpy reshape-matmul reduction),
 * string-operation restatement of stripping, decode round trips, exhaustive
 * 4^6 six-mers, brute-force BPE by a different formulation on strings <= 20
 * bases.  No function in this file is "parity unpinned".
 *
 * Class codes: A=0 C=1 G=2 T=3 N=4 UNK=5, SKIP=255 (dropped).
 */
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define CLS_N    4
#define CLS_UNK  5
#define CLS_SKIP 255

enum { MODE_SINGLE_NT = 0, MODE_KMER = 1, MODE_BPE = 2 };
enum { TAIL_PER_BASE = 0, TAIL_DROP = 1, TAIL_UNK = 2 };
enum { PAD_LEFT = 0, PAD_RIGHT = 1 };

/* Step 1 table.  PAPER.md:88 Alg. 1 l.10 (A/a, C/c, G/g, T/t, N/n), every other
 * byte -> UNK (north star; Q2), '\n' and '\r' -> SKIP (Q3).                    */
void oracle_default_lut(uint8_t lut[256]) {
    for (int b = 0; b < 256; ++b) lut[b] = CLS_UNK;
    lut['A'] = lut['a'] = 0;
    lut['C'] = lut['c'] = 1;
    lut['G'] = lut['g'] = 2;
    lut['T'] = lut['t'] = 3;
    lut['N'] = lut['n'] = CLS_N;
    lut['\n'] = CLS_SKIP;
    lut['\r'] = CLS_SKIP;
}

/* Step 1: walk one record left to right; returns the number of kept classes
 * written to cls (capacity >= len).  SURVEY.md 8(c) step 1, Q3-Q5.             */
int64_t oracle_strip(const uint8_t *rec, int64_t len, const uint8_t lut[256], int strip_headers, uint8_t *cls) {
    int64_t n = 0, i = 0;
    int line_start = 1;
    while (i < len) {
        uint8_t b = rec[i];
        if (line_start && strip_headers && b == '>') {
            while (i < len && rec[i] != '\n') ++i;   /* the header line ...            */
            if (i < len) ++i;                        /* ... up to and including '\n'   */
            line_start = 1;
            continue;
        }
        uint8_t c = lut[b];
        if (c == CLS_SKIP) {
            if (b == '\n') line_start = 1;           /* other SKIP bytes leave it as is */
        } else {
            cls[n++] = c;
            line_start = 0;
        }
        ++i;
    }
    return n;
}

/* Step 2: one ID per kept class.  PAPER.md:120 (Alg. 2 l.10).                  */
int64_t oracle_single_nt(const uint8_t *cls, int64_t n, const int32_t nt_ids[5], int32_t unk_id, int32_t *out) {
    for (int64_t i = 0; i < n; ++i) out[i] = (cls[i] <= CLS_N) ? nt_ids[cls[i]] : unk_id;
    return n;
}

/* Step 3: non-overlapping k-mers, first base most significant (Q7); a window
 * holding N or UNK -> unk_id (Q6); remainder under the tail policy (Q9).       */
int64_t oracle_kmer(const uint8_t *cls, int64_t n, int k, int32_t base_id, int32_t unk_id, int tail_policy,
                    int32_t *out) {
    int64_t t = 0, nwin = n / k;
    int64_t four_k = 1;
    for (int i = 0; i < k; ++i) four_k *= 4;
    for (int64_t j = 0; j < nwin; ++j) {
        int64_t code = 0;
        int ok = 1;
        for (int i = 0; i < k; ++i) {
            uint8_t c = cls[j * k + i];
            if (c > 3) ok = 0;
            code = code * 4 + (c & 3);
        }
        out[t++] = ok ? (int32_t)(base_id + code) : unk_id;
    }
    int64_t rem = n - nwin * k;
    if (tail_policy == TAIL_PER_BASE) {
        for (int64_t i = nwin * k; i < n; ++i)
            out[t++] = (cls[i] <= CLS_N) ? (int32_t)(base_id + four_k + cls[i]) : unk_id;
    } else if (tail_policy == TAIL_UNK) {
        if (rem > 0) out[t++] = unk_id;
    }
    return t;
}

/* Rule table for step 4: rank[left * V + right] = r for rule r, else -1,
 * V = 4 + n_merges.  Returns NULL if a rule is invalid (Q12: parts must be
 * earlier tokens, pairs unique).                                               */
int32_t *oracle_bpe_table_create(const int32_t *merges, int32_t n_merges) {
    int64_t V = 4 + (int64_t)n_merges;
    int32_t *rank = (int32_t *)malloc((size_t)(V * V) * sizeof(int32_t));
    if (!rank) return NULL;
    for (int64_t i = 0; i < V * V; ++i) rank[i] = -1;
    for (int32_t r = 0; r < n_merges; ++r) {
        int64_t L = merges[2 * r], R = merges[2 * r + 1];
        if (L < 0 || R < 0 || L >= 4 + r || R >= 4 + r || rank[L * V + R] != -1) { free(rank); return NULL; }
        rank[L * V + R] = r;
    }
    return rank;
}
void oracle_bpe_table_destroy(int32_t *rank) { free(rank); }

/* Step 4: cut at every class >= 4 (each emits n_id or unk_id, Q13); inside each
 * maximal ACGT run repeat { lowest-rank adjacent pair with a rule; replace every
 * occurrence left to right without overlap } until no pair has a rule (Q11).   */
int64_t oracle_bpe(const uint8_t *cls, int64_t n, const int32_t *rank, int32_t n_merges,
                   int32_t base_id, int32_t n_id, int32_t unk_id, int32_t *out) {
    int64_t V = 4 + (int64_t)n_merges, t = 0, i = 0;
    int32_t *seq = (int32_t *)malloc((size_t)(n > 0 ? n : 1) * sizeof(int32_t));
    while (i < n) {
        if (cls[i] >= CLS_N) { out[t++] = (cls[i] == CLS_N) ? n_id : unk_id; ++i; continue; }
        int64_t m = 0;
        while (i < n && cls[i] < CLS_N) seq[m++] = cls[i++];
        for (;;) {
            int32_t best = -1;
            for (int64_t j = 0; j + 1 < m; ++j) {
                int32_t r = rank[(int64_t)seq[j] * V + seq[j + 1]];
                if (r >= 0 && (best < 0 || r < best)) best = r;
            }
            if (best < 0) break;
            int64_t w = 0;
            for (int64_t j = 0; j < m;) {
                if (j + 1 < m && rank[(int64_t)seq[j] * V + seq[j + 1]] == best) { seq[w++] = 4 + best; j += 2; }
                else seq[w++] = seq[j++];
            }
            m = w;
        }
        for (int64_t j = 0; j < m; ++j) out[t++] = base_id + seq[j];
    }
    free(seq);
    return t;
}

/* Steps 1-5 over a batch: records [offsets[r], offsets[r+1]); ids (capacity >=
 * offsets[n_records] - offsets[0]) and out_offsets[n_records + 1] (exclusive
 * prefix sum of per-record token counts, total in the last entry).
 * Returns the total token count, or -1 on allocation failure.                  */
int64_t oracle_encode(const uint8_t *bytes, const int64_t *offsets, int64_t n_records,
                      int mode, int k, int tail_policy, int strip_headers, const uint8_t lut[256],
                      const int32_t nt_ids[5], int32_t base_id, int32_t n_id, int32_t unk_id,
                      const int32_t *rank, int32_t n_merges,
                      int32_t *ids, int64_t *out_offsets) {
    int64_t maxlen = 0, t = 0;
    for (int64_t r = 0; r < n_records; ++r)
        if (offsets[r + 1] - offsets[r] > maxlen) maxlen = offsets[r + 1] - offsets[r];
    uint8_t *cls = (uint8_t *)malloc((size_t)(maxlen > 0 ? maxlen : 1));
    if (!cls) return -1;
    out_offsets[0] = 0;
    for (int64_t r = 0; r < n_records; ++r) {
        int64_t n = oracle_strip(bytes + offsets[r], offsets[r + 1] - offsets[r], lut, strip_headers, cls);
        if (mode == MODE_SINGLE_NT)  t += oracle_single_nt(cls, n, nt_ids, unk_id, ids + t);
        else if (mode == MODE_KMER)  t += oracle_kmer(cls, n, k, base_id, unk_id, tail_policy, ids + t);
        else                         t += oracle_bpe(cls, n, rank, n_merges, base_id, n_id, unk_id, ids + t);
        out_offsets[r + 1] = t;
    }
    free(cls);
    return t;
}

/* Step 6: row r holds record r's first m = min(tokens, seq_len) IDs; LEFT puts
 * them at columns [seq_len - m, seq_len) (right-aligned), RIGHT at
 * [0, m); other columns pad_id; mask is 1 exactly on the m kept columns (Q14-16). */
void oracle_pad(const int32_t *ids, const int64_t *out_offsets, int64_t n_records,
                int32_t seq_len, int pad_side, int32_t pad_id, int32_t *batch_ids, uint8_t *mask) {
    for (int64_t r = 0; r < n_records; ++r) {
        int64_t tok = out_offsets[r + 1] - out_offsets[r];
        int64_t m = tok < seq_len ? tok : seq_len;
        int64_t col0 = (pad_side == PAD_LEFT) ? seq_len - m : 0;
        for (int64_t c = 0; c < seq_len; ++c) { batch_ids[r * seq_len + c] = pad_id; mask[r * seq_len + c] = 0; }
        for (int64_t j = 0; j < m; ++j) {
            batch_ids[r * seq_len + col0 + j] = ids[out_offsets[r] + j];
            mask[r * seq_len + col0 + j] = 1;
        }
    }
}
