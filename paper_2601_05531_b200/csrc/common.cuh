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
#ifndef DTK_NT
#define DTK_NT 256
#endif
constexpr int NT = DTK_NT;              // threads per CTA of the encode kernel
constexpr int LB = 64;                  // input bytes per thread
constexpr int TB = NT * LB;             // input bytes per sub-tile (16 KiB)
constexpr int S_MAX = 4;                // sub-tiles per super-tile (the unit of the chained scan), at most

// ---- scan protocol -------------------------------------------------------------------
enum : uint32_t { ST_EMPTY = 0, ST_AGG = 1, ST_INCL = 2 };
enum : uint32_t { LS_LINE_START = 0, LS_IN_LINE = 1, LS_IN_HEADER = 2 };
enum : uint32_t { LK_NONE = 0, LK_SUMMARY = 1, LK_FINAL = 2 };
constexpr int SPIN_LIMIT = 1 << 22;     // bounded spin: a broken chain sets the status word instead of hanging

// One 64-byte descriptor per super-tile, made of self-validating words: every 16-byte word carries the tag
// (generation << 2 | ST_*) of the call that wrote it, is written with one 16-byte store and read with one
// 16-byte load that bypasses L1, so no fence or acquire/release pair is needed and the scratch never needs
// clearing between calls.  a0/a1 describe the super-tile alone (aggregate), i0/i1 the whole prefix up to and
// including it (inclusive).  Class tails hold 3 bits per class, newest class lowest.
//   a0 = { tagA, first_kept, last_kept, closed | has_event << 31 }
//   a1 = { tagA, tail_cnt | tail_hi10 << 4, tail_lo32, 0 }
//   i0 = { tagI, T lo, T hi, open_r | tail_cnt << 4 | tail_hi10 << 8 }
//   i1 = { tagI, open_q lo, open_q hi, tail_lo32 }
// The line-state chain has one 4-byte word per super-tile in an array of its own:
//   ls = gen << 8 | LK_* << 2 | line state
struct __align__(16) TileDesc {
    uint4 a0;
    uint4 a1;
    uint4 i0;
    uint4 i1;
};
static_assert(sizeof(TileDesc) == 64, "TileDesc layout");

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
    int32_t fast_n;         // class_lut maps 'N' and 'n' to CLS_N: runs of N can be classified arithmetically too
    uint32_t kmagic;        // floor(2^32 / k) + 1 (k >= 2): n / k == umulhi(n, kmagic) for n < 2^28
    // table-driven k-mer ids (Alg. 1 l.18-22, kmer_lut[0..5^k-1]); both null: the base-4 closed form
    const int32_t *kmer_lut;    // [5^k] id of every base-5 window code (digit 4 = N or any other kept byte)
    const int32_t *remap4;      // [4^k] kmer_lut[code5(code4)]: the id of every window of A, C, G, T
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
    TileDesc *descs;              // [n_tiles]
    TileDesc *gdescs;             // [n_tiles / 32 + 1] group aggregates (a0 / a1 only) of the two-level look-back
    uint32_t *ls;                 // [n_tiles] line-state chain words
    int64_t *first_rec;           // [n_tiles + 1]: first r in [0, n_rec] whose position is >= tile * S * TB (n_rec + 1 if none)
    int32_t *rec_k;               // [n_rec + 1] scratch: kept bases of the super-tile before each record start (many-starts path)
    unsigned long long *ticket;   // tile ticket counter
    unsigned long long ticket_base;
    uint32_t *status;             // device-mapped host status word
    unsigned long long *prof;     // phase timers (debug builds with -DDTK_PROF only)
    const uint32_t *run_if;       // non-null: the chained-scan encoder runs only if *run_if != 0 (set by the regular-layout fast path)
    uint32_t gen;
    int32_t n_tiles;              // super-tiles
    int32_t S;                    // sub-tiles per super-tile (1..S_MAX)
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

__device__ __forceinline__ int64_t rec_pos(const EncArgs &A, int64_t r) { return A.rec_off[r] - A.off_bias + A.mis; }

// table-driven id of one window: `code` = its k base-4 digits (first base most significant), `flags` = k bits, set
// where the base is not A, C, G, T (its digit then counts as 4)
__device__ __forceinline__ int32_t kmer_table_id(const EncParams &P, uint32_t code, uint32_t flags, int k) {
    if (!flags) return __ldg(P.remap4 + code);
    uint32_t c5 = 0;
    for (int i = k - 1; i >= 0; --i) c5 = c5 * 5u + (((flags >> i) & 1u) ? 4u : ((code >> (2 * i)) & 3u));
    return __ldg(P.kmer_lut + c5);
}

// the same, out of line: for the token-at-a-time paths of the per-k kernels, whose loops are sensitive to their footprint
__device__ __noinline__ int32_t kmer_table_id_cold(const EncParams &P, uint32_t code, uint32_t flags, int k) {
    return kmer_table_id(P, code, flags, k);
}

// n / k for 0 <= n < 2^28 without a divide (k = 1 passes through)
__device__ __forceinline__ uint32_t div_k(uint32_t n, const EncParams &P) {
    return P.k == 1 ? n : __umulhi(n, P.kmagic);
}

struct QR { int64_t q; int32_t r; };     // n = q * k + r, 0 <= r < k

__device__ __forceinline__ QR qr_of(uint32_t n, const EncParams &P) {
    QR x; const uint32_t q = div_k(n, P); x.q = q; x.r = (int32_t)(n - q * (uint32_t)P.k); return x;
}
__device__ __forceinline__ QR qr_add(QR a, QR b, int k) {
    QR x; int r = a.r + b.r; int c = r >= k;
    x.q = a.q + b.q + c; x.r = r - (c ? k : 0);
    return x;
}
// tokens emitted for the n mod k = r trailing bases of a record that closes
__device__ __forceinline__ int tail_tokens(int r, const EncParams &P) {
    if (P.mode != MODE_KMER || P.tail_policy == TAIL_PER_BASE) return r;
    return (P.tail_policy == TAIL_UNK && r != 0) ? 1 : 0;
}
// tokens a record of x kept bases emits (k-mer: windows + tail policy; single-nt: k = 1, r = 0)
__device__ __forceinline__ int64_t qr_tokens(QR x, const EncParams &P) { return x.q + tail_tokens(x.r, P); }
__device__ __forceinline__ int tok_count32(int n, const EncParams &P) {
    if (P.mode != MODE_KMER) return n;
    const int w = (int)div_k((uint32_t)n, P), r = n - w * P.k;
    return w + tail_tokens(r, P);
}

}  // namespace dtk
