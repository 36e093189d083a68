// common.cuh -- shared device-side definitions for the DNATok sm_100a kernels.
//
// Scan state and tile summaries for the single-pass (decoupled look-back) encoder.
// See DESIGN.md "Kernels" for the derivation; SURVEY.md section 7 hard parts 2-4 for why
// a single pass over flat byte tiles is needed to stay under the HBM roofline.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace dtk {

// ---- class codes (include/dnatok.h) -------------------------------------------------
constexpr uint32_t CLS_N = 4, CLS_UNK = 5, CLS_SKIP = 255;

// ---- modes ---------------------------------------------------------------------------
enum : int { MODE_SINGLE_NT = 0, MODE_KMER = 1, MODE_BPE = 2 };
enum : int { TAIL_PER_BASE = 0, TAIL_DROP = 1, TAIL_UNK = 2 };

// ---- tile geometry -------------------------------------------------------------------
constexpr int NT = 256;                 // threads per CTA

// ---- scan protocol -------------------------------------------------------------------
enum : uint32_t { ST_EMPTY = 0, ST_AGG = 1, ST_INCL = 2 };
enum : uint32_t { LS_LINE_START = 0, LS_IN_LINE = 1, LS_IN_HEADER = 2 };
constexpr int SPIN_LIMIT = 1 << 22;     // bounded spin: a broken chain sets the status word instead of hanging

// One descriptor per tile, made of self-validating 16-byte words: every word carries the tag
// (generation << 2 | ST_*) of the call that wrote it, is written with one 16-byte store and read with one
// 16-byte load that bypasses L1, so no fence or acquire/release pair is needed and the scratch never needs
// clearing between calls.  a0/a1 describe the tile alone (aggregate), i0..i2 the whole prefix up to and
// including the tile (inclusive).  Kept-base counts that can span many tiles are held as (quotient,
// remainder) by k so that composing them never divides.
struct __align__(16) TileDesc {
    uint4 a0;               // tag, first_kept, last_kept, closed_tokens
    uint4 a1;               // tag, tail_cnt | has_event << 8, tail lo, tail hi
    uint4 i0;               // tag, ptail_cnt | open_r << 8, T lo, T hi
    uint4 i1;               // tag, 0, open_q lo, open_q hi
    uint4 i2;               // tag, 0, ptail lo, ptail hi
    uint32_t l_word;        // gen<<8 | has_reset<<2 | exit_if_line_start   (line-state summary)
    uint32_t l_incl;        // gen<<8 | exit line state                     (line-state inclusive)
    uint32_t pad_[2];
};
static_assert(sizeof(TileDesc) == 96, "TileDesc layout");

struct QR { int64_t q; int32_t r; };     // n = q * k + r, 0 <= r < k

// aggregate of one tile or of a run of tiles:
//   first: kept bases before the first record start (all of them if no event)
//   last:  kept bases after the last record start   (all of them if no event)
//   closed: tokens of records that open AND close inside
//   tail: last tail_cnt (<= k-1) kept classes of the last segment, 4 bits each, newest lowest
struct Agg {
    QR first, last; int64_t closed;
    uint64_t tail; uint32_t tail_cnt; uint32_t has_event;
};
// inclusive prefix: T = out_offsets[] of the record open at the boundary, open = its kept bases so far
struct Prefix {
    int64_t T; QR open; uint64_t tail; uint32_t tail_cnt;
};

// ---- encoder parameters (device copy of the create-time spec) -------------------------
struct EncParams {
    int32_t mode;           // MODE_SINGLE_NT | MODE_KMER (BPE runs the class-stream pass as SINGLE_NT)
    int32_t k;
    int32_t tail_policy;
    int32_t strip_headers;
    int32_t unk_id, base_id;
    int32_t nt_ids[5];
    int32_t four_k;         // 4^k (KMER; fits: k <= 15)
    int32_t fast_lut;       // class_lut maps ACGTacgt to 0..3 like the default: arithmetic classification is exact for them
};

struct EncArgs {
    const uint8_t *bytes_al;      // 16-byte aligned-down input pointer
    int64_t mis;                  // d_bytes - bytes_al (0..15); "position" p addresses bytes_al[p]
    int64_t p_end;                // mis + n_bytes
    const int64_t *rec_off;       // [n_rec + 1]
    int64_t n_rec;
    int64_t off_bias;             // position of record offset v is v - off_bias + mis
    void *ids;                    // output ids (uint8 / int16 / int32)
    int64_t ids_cap;
    int64_t *out_off;             // [n_rec + 1]
    int64_t out_bias;             // added to every out_off value and id position (0)
    const uint8_t *lut;           // [256] device
    TileDesc *descs;
    unsigned long long *ticket;   // tile ticket counter
    unsigned long long ticket_base;
    uint32_t *status;             // device-mapped host status word
    uint32_t gen;
    int32_t n_tiles;
    EncParams prm;
};

// ---- small helpers --------------------------------------------------------------------
__device__ __forceinline__ uint32_t ld_vol32(const uint32_t *p) {
    uint32_t v;
    asm volatile("ld.volatile.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_vol32(uint32_t *p, uint32_t v) {
    asm volatile("st.volatile.global.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}
__device__ __forceinline__ uint4 ld_vol128(const uint4 *p) {
    uint4 v;
    asm volatile("ld.volatile.global.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_vol128(uint4 *p, uint4 v) {
    asm volatile("st.volatile.global.v4.u32 [%0], {%1, %2, %3, %4};" ::"l"(p), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
}

__device__ __forceinline__ QR qr_of(int n, int k) { QR x; x.q = n / k; x.r = n - (int)x.q * k; return x; }
__device__ __forceinline__ QR qr_add(QR a, QR b, int k) {
    QR x; int r = a.r + b.r; int c = r >= k;
    x.q = a.q + b.q + c; x.r = r - (c ? k : 0);
    return x;
}
// tokens a record of x kept bases emits (k-mer: windows + tail policy; single-nt: k = 1, r = 0)
__device__ __forceinline__ int64_t qr_tokens(QR x, const EncParams &P) {
    if (P.mode != MODE_KMER || P.tail_policy == TAIL_PER_BASE) return x.q + x.r;
    return x.q + ((P.tail_policy == TAIL_UNK && x.r != 0) ? 1 : 0);
}
__device__ __forceinline__ int tok_count32(int n, const EncParams &P) {
    if (P.mode != MODE_KMER) return n;
    int w = n / P.k, r = n - w * P.k;
    if (P.tail_policy == TAIL_PER_BASE) return w + r;
    if (P.tail_policy == TAIL_UNK) return w + (r != 0);
    return w;
}

__device__ __forceinline__ uint64_t nib_mask(uint32_t n) { return n >= 16 ? ~0ull : ((1ull << (4 * n)) - 1); }

// tail of (a followed by b), truncated to kmax nibbles
__device__ __forceinline__ void tail_concat(uint64_t a, uint32_t an, uint64_t b, uint32_t bn, uint32_t kmax,
                                            uint64_t &o, uint32_t &on) {
    uint32_t n = an + bn; if (n > kmax) n = kmax;
    uint64_t v = (bn >= 16 ? 0ull : (a << (4 * bn))) | b;
    o = v & nib_mask(n); on = n;
}

// A (earlier) followed by B (later)
__device__ __forceinline__ Agg agg_compose(const Agg &A, const Agg &B, const EncParams &P) {
    Agg R; const uint32_t kmax = (uint32_t)(P.k - 1);
    if (!B.has_event) {
        if (B.tail_cnt >= kmax) { R.tail = B.tail; R.tail_cnt = B.tail_cnt; }
        else tail_concat(A.tail, A.tail_cnt, B.tail, B.tail_cnt, kmax, R.tail, R.tail_cnt);
        if (!A.has_event) {
            R.first = R.last = qr_add(A.first, B.first, P.k); R.closed = 0; R.has_event = 0;
        } else {
            R.first = A.first; R.closed = A.closed; R.last = qr_add(A.last, B.first, P.k); R.has_event = 1;
        }
    } else {
        R.tail = B.tail; R.tail_cnt = B.tail_cnt; R.last = B.last; R.has_event = 1;
        if (!A.has_event) { R.first = qr_add(A.first, B.first, P.k); R.closed = B.closed; }
        else { R.first = A.first; R.closed = A.closed + qr_tokens(qr_add(A.last, B.first, P.k), P) + B.closed; }
    }
    return R;
}

__device__ __forceinline__ Prefix prefix_apply(const Prefix &X, const Agg &A, const EncParams &P) {
    Prefix R; const uint32_t kmax = (uint32_t)(P.k - 1);
    if (!A.has_event) {
        R.T = X.T; R.open = qr_add(X.open, A.first, P.k);
        if (A.tail_cnt >= kmax) { R.tail = A.tail; R.tail_cnt = A.tail_cnt; }
        else tail_concat(X.tail, X.tail_cnt, A.tail, A.tail_cnt, kmax, R.tail, R.tail_cnt);
    } else {
        R.T = X.T + qr_tokens(qr_add(X.open, A.first, P.k), P) + A.closed;
        R.open = A.last; R.tail = A.tail; R.tail_cnt = A.tail_cnt;
    }
    return R;
}

}  // namespace dtk
