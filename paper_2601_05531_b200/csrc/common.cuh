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
constexpr int SPAN = 32;                // bytes per thread = one bitmap word
constexpr int TB = NT * SPAN;           // tile bytes (8 KiB)
constexpr int PEND_MAX = 16;            // slots in front of the compact class array for carried bases

// ---- scan protocol -------------------------------------------------------------------
enum : uint32_t { ST_EMPTY = 0, ST_AGG = 1, ST_INCL = 2 };
enum : uint32_t { LS_LINE_START = 0, LS_IN_LINE = 1, LS_IN_HEADER = 2 };
constexpr uint32_t STATUS_ECAPACITY = 1u, STATUS_ESTATE = 2u;
constexpr int SPIN_LIMIT = 1 << 22;     // bounded spin: a broken chain sets STATUS_ESTATE instead of hanging

// One descriptor per tile.  Aggregate fields describe the tile alone; inclusive fields
// describe the whole prefix up to and including the tile.  Both are published with a
// release store of `status` / `l_word` / `l_incl` tagged by the call's generation number,
// so the scratch never needs clearing between calls.
struct __align__(16) TileDesc {
    uint32_t l_word;        // gen<<8 | has_reset<<2 | exit_if_line_start   (line-state summary)
    uint32_t l_incl;        // gen<<8 | exit line state                     (line-state inclusive)
    uint32_t status;        // gen<<2 | ST_*
    uint32_t has_event;     // a record starts (or the last record ends) inside the tile
    int32_t  first_kept;    // kept bases before the first event (all of them if no event)
    int32_t  last_kept;     // kept bases after the last event   (all of them if no event)
    int64_t  closed_tokens; // tokens of records that open AND close inside the tile
    uint64_t tail;          // last tail_cnt kept classes of the last segment, 4 bits each, newest lowest
    uint32_t tail_cnt;      // min(k-1, kept in last segment)
    uint32_t pad_;
    // inclusive prefix after this tile
    int64_t  T;             // out_offsets[] of the record open at the tile's end
    int64_t  open_n;        // kept bases of that record so far
    uint64_t ptail;         // its last ptail_cnt kept classes
    uint32_t ptail_cnt;     // min(k-1, open_n)
    uint32_t pad2_;
};
static_assert(sizeof(TileDesc) == 80, "TileDesc layout");

struct Agg {                // composed aggregate (64-bit counters: a record may span many tiles)
    int64_t first_kept, last_kept, closed_tokens;
    uint64_t tail; uint32_t tail_cnt; uint32_t has_event;
};
struct Prefix {
    int64_t T, open_n; uint64_t tail; uint32_t tail_cnt;
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
__device__ __forceinline__ uint32_t ld_acquire(const uint32_t *p) {
    uint32_t v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_release(uint32_t *p, uint32_t v) {
    asm volatile("st.release.gpu.global.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}

__device__ __forceinline__ int64_t tok_count(int64_t n, const EncParams &P) {
    if (P.mode != MODE_KMER) return n;
    int64_t w = n / P.k, r = n - w * P.k;
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

// acc = A (earlier) composed with acc (later)
__device__ __forceinline__ Agg agg_compose(const Agg &A, const Agg &B, const EncParams &P) {
    Agg R; uint32_t kmax = (uint32_t)(P.k - 1);
    if (!B.has_event) {
        tail_concat(A.tail, A.tail_cnt, B.tail, B.tail_cnt, kmax, R.tail, R.tail_cnt);
        if (!A.has_event) {
            R.first_kept = R.last_kept = A.first_kept + B.first_kept; R.closed_tokens = 0; R.has_event = 0;
        } else {
            R.first_kept = A.first_kept; R.closed_tokens = A.closed_tokens;
            R.last_kept = A.last_kept + B.first_kept; R.has_event = 1;
        }
    } else {
        R.tail = B.tail; R.tail_cnt = B.tail_cnt; R.last_kept = B.last_kept; R.has_event = 1;
        if (!A.has_event) { R.first_kept = A.first_kept + B.first_kept; R.closed_tokens = B.closed_tokens; }
        else {
            R.first_kept = A.first_kept;
            R.closed_tokens = A.closed_tokens + tok_count(A.last_kept + B.first_kept, P) + B.closed_tokens;
        }
    }
    return R;
}

__device__ __forceinline__ Prefix prefix_apply(const Prefix &X, const Agg &A, const EncParams &P) {
    Prefix R; uint32_t kmax = (uint32_t)(P.k - 1);
    if (!A.has_event) {
        R.T = X.T; R.open_n = X.open_n + A.first_kept;
        tail_concat(X.tail, X.tail_cnt, A.tail, A.tail_cnt, kmax, R.tail, R.tail_cnt);
    } else {
        R.T = X.T + tok_count(X.open_n + A.first_kept, P) + A.closed_tokens;
        R.open_n = A.last_kept; R.tail = A.tail; R.tail_cnt = A.tail_cnt;
    }
    return R;
}

}  // namespace dtk
