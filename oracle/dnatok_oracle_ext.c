/*
 * dnatok_oracle_ext.c -- plain CPU definitions of the SURVEY.md 8(f) operations (the rows marked "next"):
 * f1 table-driven k-mer IDs, f2 embedding gather + micro-batch rule, f3 decode and reverse complement,
 * f4 int32 -> int64 widening of an ID matrix.  TEST INFRASTRUCTURE ONLY, same rules as dnatok_oracle.c:
 * only tests/, __graft_entry__.smoke() and bench.py's CPU legs may build, load or call it; it shares nothing
 * with the CUDA path.  One byte / one token at a time, in the order the cited passages state.
 *
 * Pins (tests/test_oracle_ext.py): hand-worked values, Python string operations for the reverse complement
 * (reverse + translate), involution RC(RC(x)) = x, decode(encode(s)) = upper(stripped s) on N-free input,
 * base-5 closed form with numpy, a k-mer table that reproduces the base-4 closed form, the paper's printed
 * micro-batch formula evaluated by hand, numpy fancy indexing for the gather.  No function is "parity unpinned".
 */
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define CLS_N    4
#define CLS_UNK  5
enum { MODE_SINGLE_NT = 0, MODE_KMER = 1, MODE_BPE = 2 };
enum { TAIL_PER_BASE = 0, TAIL_DROP = 1, TAIL_UNK = 2 };

/* ---- f1: Alg. 1 l.18-22 (k-mer structure "length k, stride k", base5_lut[0..255] -> {0..4},
 * kmer_lut[0..5^k-1]); Alg. 2 l.7-8 (MapKmer).  Window j of the kept classes is turned into the
 * base-5 number sum_i digit_i * 5^(k-1-i) (first base most significant, as Q7), digit = class for A,C,G,T and 4
 * for N and for every other kept byte (PAPER.md:88 l.27: the table starts out as N's entry for every byte); the ID
 * is kmer_lut[code].  The table, not the encoder, decides what a window holding N becomes.  The n mod k trailing
 * bases: PER_BASE -> nt_ids[class] (UNK byte -> unk_id), DROP -> nothing, UNK -> one unk_id.                      */
int64_t oracle_kmer_table(const uint8_t *cls, int64_t n, int k, const int32_t *kmer_lut, const int32_t nt_ids[5],
                          int32_t unk_id, int tail_policy, int32_t *out) {
    int64_t t = 0, nwin = n / k;
    for (int64_t j = 0; j < nwin; ++j) {
        int64_t code = 0;
        for (int i = 0; i < k; ++i) {
            uint8_t c = cls[j * k + i];
            code = code * 5 + (c < CLS_N ? c : 4);
        }
        out[t++] = kmer_lut[code];
    }
    if (tail_policy == TAIL_PER_BASE) {
        for (int64_t i = nwin * k; i < n; ++i) out[t++] = (cls[i] <= CLS_N) ? nt_ids[cls[i]] : unk_id;
    } else if (tail_policy == TAIL_UNK) {
        if (n - nwin * k > 0) out[t++] = unk_id;
    }
    return t;
}

/* ---- f2: PAPER.md:66-72 (section 2 notation: IDs [B x T'] -> embeddings [B x T' x D]), Alg. 2 l.17 and
 * PAPER.md:181 (micro-batch size b = min(B_emb, max(1, floor(M / T'))), M = 1,048,576 tokens per call).            */
int64_t oracle_microbatch_rows(int64_t b_emb, int64_t m_tokens, int64_t t_len) {
    int64_t q = t_len > 0 ? m_tokens / t_len : m_tokens;
    if (q < 1) q = 1;
    return b_emb < q ? b_emb : q;
}
/* out[i] = table[ids[i]] for every token i, rows of row_bytes bytes; an ID outside [0, vocab) gives a zero row.     */
void oracle_embed(const int32_t *ids, int64_t n_tokens, const uint8_t *table, int64_t vocab, int64_t row_bytes,
                  uint8_t *out) {
    for (int64_t i = 0; i < n_tokens; ++i) {
        if (ids[i] >= 0 && ids[i] < vocab) memcpy(out + i * row_bytes, table + (int64_t)ids[i] * row_bytes, (size_t)row_bytes);
        else memset(out + i * row_bytes, 0, (size_t)row_bytes);
    }
}

/* ---- f3: PAPER.md:325-327 (section 4.5.4, reverse complement on device as future work).  Each record is reversed
 * and every byte replaced by its complement: A<->T, C<->G, U->A, the IUPAC codes R<->Y, K<->M, B<->V, D<->H,
 * S, W, N unchanged, case kept; every other byte (line breaks included) unchanged.                                   */
static uint8_t comp_byte(uint8_t b) {
    static const char from[] = "ACGTURYKMBVDHSWNacgturykmbvdhswn";
    static const char to[]   = "TGCAAYRMKVBHDSWNtgcaayrmkvbhdswn";
    for (int i = 0; from[i]; ++i) if ((uint8_t)from[i] == b) return (uint8_t)to[i];
    return b;
}
void oracle_revcomp(const uint8_t *bytes, const int64_t *offsets, int64_t n_records, uint8_t *out) {
    for (int64_t r = 0; r < n_records; ++r) {
        int64_t a = offsets[r], e = offsets[r + 1];
        for (int64_t j = 0; j < e - a; ++j) out[a + j] = comp_byte(bytes[e - 1 - j]);
    }
}

/* ---- f3: PAPER.md:315-317 (section 4.5.2: decoding through an inverse vocabulary table).  Every token is replaced
 * by its spelling in upper case; pad_id tokens are skipped.
 *   single-nt: nt_ids[c] -> "ACGTN"[c]; any other ID -> 'N'
 *   k-mer:     base_id + code (code < 4^k) -> its k bases, first base most significant (Q7); base_id + 4^k + c
 *              (c < 5, the per-base tail IDs of Q9) -> "ACGTN"[c]; any other ID (UNK: a window that held N, Q6) -> k x 'N'
 *   BPE:       n_id -> 'N'; base_id + t (t < 4 + n_merges) -> spelling(t), spelling of a base is itself and
 *              spelling(4 + r) = spelling(left_r) spelling(right_r); any other ID -> 'N'
 * byte_offsets[n_records + 1] gets the exclusive prefix sum of the decoded record lengths.  Returns the total number
 * of bytes, or -1 if it exceeds cap.                                                                                */
static int64_t spell(const int32_t *merges, int32_t t, uint8_t *out, int64_t pos, int64_t cap) {
    if (t < 4) { if (pos < cap) out[pos] = (uint8_t)"ACGT"[t]; return pos + 1; }
    pos = spell(merges, merges[2 * (t - 4)], out, pos, cap);
    return spell(merges, merges[2 * (t - 4) + 1], out, pos, cap);
}
int64_t oracle_decode(const int32_t *ids, const int64_t *out_offsets, int64_t n_records, int mode, int k,
                      const int32_t nt_ids[5], int32_t base_id, int32_t n_id, int32_t unk_id, int32_t pad_id,
                      const int32_t *merges, int32_t n_merges, uint8_t *out, int64_t cap, int64_t *byte_offsets) {
    (void)unk_id;
    int64_t pos = 0, four_k = 1;
    for (int i = 0; i < k; ++i) four_k *= 4;
    byte_offsets[0] = 0;
    for (int64_t r = 0; r < n_records; ++r) {
        for (int64_t j = out_offsets[r]; j < out_offsets[r + 1]; ++j) {
            int32_t id = ids[j];
            if (id == pad_id) continue;
            if (mode == MODE_SINGLE_NT) {
                uint8_t ch = 'N';
                for (int c = 0; c < 5; ++c) if (id == nt_ids[c]) { ch = (uint8_t)"ACGTN"[c]; break; }
                if (pos < cap) out[pos] = ch;
                ++pos;
            } else if (mode == MODE_KMER) {
                int64_t code = (int64_t)id - base_id;
                if (code >= 0 && code < four_k) {
                    for (int i = 0; i < k; ++i) {
                        int64_t d = code;
                        for (int s = 0; s < k - 1 - i; ++s) d /= 4;
                        if (pos < cap) out[pos] = (uint8_t)"ACGT"[d % 4];
                        ++pos;
                    }
                } else if (code >= four_k && code < four_k + 5) {
                    if (pos < cap) out[pos] = (uint8_t)"ACGTN"[code - four_k];
                    ++pos;
                } else {
                    for (int i = 0; i < k; ++i) { if (pos < cap) out[pos] = 'N'; ++pos; }
                }
            } else {
                int64_t t = (int64_t)id - base_id;
                if (id == n_id || t < 0 || t >= 4 + (int64_t)n_merges) { if (pos < cap) out[pos] = 'N'; ++pos; }
                else pos = spell(merges, (int32_t)t, out, pos, cap);
            }
        }
        byte_offsets[r + 1] = pos;
    }
    return pos <= cap ? pos : -1;
}

/* ---- f4: PAPER.md:82 (section 2.2, IDs path: "32-bit + on-device cast" -- an int32 ID matrix widened to int64).       */
void oracle_widen(const int32_t *ids, int64_t n, int64_t *out) {
    for (int64_t i = 0; i < n; ++i) out[i] = (int64_t)ids[i];
}
