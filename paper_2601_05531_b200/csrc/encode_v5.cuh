// encode_v5.cuh -- single-pass classify + strip + {single-nt | k-mer} + CSR offsets over chained, software-pipelined
// SUPER-TILES.  This is the encoder of specs that DROP bytes (a SKIP class and / or header stripping); specs that keep
// every byte run the no-scan encoder of encode_v7.cuh.  (Everything here lives in dtk::v5: the two encoders share
// common.cuh only.)
//
// One persistent CTA (256 threads, 4 per SM) claims flat super-tiles of S x 16 KiB input bytes in order (atomic
// ticket, fetched one super-tile ahead together with its record range, its entry line state and an L2 prefetch).
// The super-tile is the unit of the chained scan (decoupled look-back).  The CTA works on two super-tiles at a
// time: while the predecessors of super-tile A finish, it already runs the sub-tile loop of the next one, B, into
// the second kept-base stream buffer, publishes B's aggregate, and only then looks back for A and emits A:
//     loop(B) -> publish aggregate(B) -> look-back(A), publish inclusive(A) -> emit(A) -> A := B
// Sub-tile loop (two block barriers per 16 KiB, no one-warp section); each thread owns 64 contiguous input bytes,
// loaded straight into registers with four 16-byte loads:
//   P1 classify ("256-entry LUT"; Alg. 1): ACGT in either case is recognised
//      arithmetically on four bytes per 32-bit register -- the 2-bit code is ASCII bits 1..2, validity is one
//      masked compare -- and gathered into per-thread bit planes by a multiply (code plane: 2 bits x 64 bases,
//      exception plane: 1 bit x 64).  Every byte the arithmetic does not prove to be ACGT goes through the
//      256-entry LUT in shared memory: the table remains the specification.  Line state (LINE_START / IN_LINE /
//      IN_HEADER) is summarised per thread as a function of the entry state and scanned across the warp.
//   P2 header mask, keep mask, in-register compaction of the planes (runs of dropped bytes deleted), warp scan of
//      the kept counts.
//   P3 planes appended to the super-tile's kept-base stream in shared memory (2-bit base-4 digits, MSB first, plus
//      a "not ACGT" flag plane); the kept-base index of every record start inside the warp's bytes is noted.
// Entry line state of a super-tile: read off the 128 bytes in front of it when they hold a newline or the record's
//   start (always, for wrapped FASTA); otherwise the loop runs under the assumption IN_LINE, the state comes from a
//   chain of its own (one word per super-tile) and the rare super-tiles where it matters are redone.
// Look-back (warp 0): windows of 32 predecessors are folded in parallel; a window without an inclusive prefix is
//   folded into a running aggregate and the walk continues further back, so no super-tile ever waits for a
//   predecessor's look-back, only for its aggregate.
// Emission: tokens are cut from the stream in groups of 16 output bytes: one funnel-shift alignment per group,
//   windows at compile-time offsets, one 16-byte store straight to ids_out.
// Input bytes are read from HBM exactly once and ids written exactly once.
#pragma once
#include "common.cuh"

namespace dtk {
namespace v5 {

constexpr int NW = NT / 32;
static_assert(NW % 4 == 0, "warp summaries are read four at a time");
constexpr int WB = 32 * LB;                  // input bytes per warp per sub-tile (2 KiB)
constexpr int PEND = 16;                     // stream slots in front of the super-tile's kept bases (carried bases)
constexpr int STREAM_BASES = PEND + S_MAX * TB;
constexpr int SW_CODE = (STREAM_BASES / 16 + 8 + 3) & ~3;
constexpr int SW_FLAG = (STREAM_BASES / 32 + 9 + 3) & ~3;
constexpr int SW_ALL = SW_CODE + SW_FLAG;    // multiple of 4 words
constexpr int EVW = 32;                      // record starts per super-tile handled by the one-warp path
constexpr int ENT_CAP = NT + 1;              // segment-table entries per emission pass (many-starts path)
constexpr uint32_t LS_UNKNOWN = 3;

struct TileAgg {                             // aggregate of one super-tile, kept until its look-back
    int32_t fk, lk, closed, tn, ntok;        // kept before first / after last record start, tokens of records inside,
    uint32_t hasev;                          //   tail classes held, tokens of the segment table so far
    unsigned long long tail;                 // last tn classes, 3 bits each, newest lowest
};

struct Smem5 {
    uint32_t strm[2][SW_ALL];                // per buffer -- code stream: base u at word u>>4, bits 31-2(u&15), 30-2(u&15);
                                             // flag stream at + SW_CODE: base u at word u>>5, bit 31-(u&31)
    unsigned long long wk[NW][32];           // per warp: record-start bitmap of its 2 KiB (P1), then keep masks (P3)
    int32_t ent_src[ENT_CAP];                // many-starts segment table: stream position of the segment's first base
    int32_t ent_t[ENT_CAP];                  //   super-tile-relative index of its first token
    int32_t ent_nwin[ENT_CAP];               //   full windows available (tokens beyond are tail tokens)
    int32_t seg_src[2][EVW + 1];             // the same for at most EVW record starts, per buffer
    int32_t seg_t[2][EVW + 1];
    int32_t seg_nwin[2][EVW + 1];
    int32_t ev_p[2][EVW];                    // super-tile positions of the first EVW record starts (by ticket parity)
    int32_t ev_k[2][EVW];                    // kept bases before each of them (per buffer)
    uint16_t offw[NW][32];                   // per warp: exclusive kept-base prefix of each lane
    alignas(16) int32_t warp_cnt[2][NW];     // by sub-tile parity
    alignas(16) uint32_t warp_ls[2][NW];
    uint32_t ls_sub[2];                      // exit line state of the sub-tile (by sub-tile parity)
    int32_t scan_tmp[NW];
    uint8_t lut[256];
    TileAgg ag[2];                           // per buffer
    // control of the next super-tile to loop over (by ticket parity)
    int32_t c_tile[2], c_m[2];
    uint32_t c_ls[2];
    long long c_rlo[2];
    // scalars
    uint32_t t_ls, ls_in, redo;
    int32_t tok0, ntok;                      // emission: tokens of the open record's piece, tokens of the super-tile
    long long T0;                            // global index of the super-tile's first token
};
static_assert(sizeof(Smem5) <= (NT >= 256 ? 56 * 1024 * (NT / 256) : 32 * 1024), "shared memory per CTA");

// ---------------------------------------------------------------------------------------- small helpers
__device__ __forceinline__ unsigned long long bit_at(int q) { return 0x8000000000000000ull >> q; }          // q in 0..63
__device__ __forceinline__ unsigned long long from_pos(int q) { return q >= 64 ? 0ull : (~0ull >> q); }   // positions >= q
__device__ __forceinline__ int first_pos(unsigned long long m) { return m ? __clzll((long long)m) : 64; }

// k digits starting at base u (k <= 16) of the stream buffer st
__device__ __forceinline__ uint32_t code_at(const uint32_t *st, int u, int k) {
    const int b = 2 * u, w = b >> 5, s = b & 31;
    return __funnelshift_l(st[w + 1], st[w], s) >> (32 - 2 * k);
}
__device__ __forceinline__ uint32_t flags_at(const uint32_t *st, int u, int k) {    // k flag bits starting at base u
    const int w = u >> 5, s = u & 31;
    const uint32_t *f = st + SW_CODE;
    return __funnelshift_l(f[w + 1], f[w], s) >> (32 - k);
}
// class code 0..5 of base u: ACGT from the code plane; flagged bases carry digit 2 for N (what the arithmetic
// classification yields for 'N' / 'n') and digit 1 for UNK
__device__ __forceinline__ uint32_t class_at(const uint32_t *st, int u) {
    const uint32_t c = code_at(st, u, 1);
    return flags_at(st, u, 1) ? (c == 2u ? CLS_N : CLS_UNK) : c;
}

template <typename IdT>
__device__ __forceinline__ void store_id(const EncArgs &A, int64_t idx, int32_t id) {
    if (idx < A.ids_cap) reinterpret_cast<IdT *>(A.ids)[idx] = (IdT)id;
    else A.status[0] = 1u;
}

// ---- line state as a function: a summary (hr, x) maps the entry state e to hr ? x : (e == LINE_START ? x : e) ----
__device__ __forceinline__ uint32_t ls_apply(uint32_t hr, uint32_t x, uint32_t e) { return hr ? x : (e == LS_LINE_START ? x : e); }

// ---- classification -----------------------------------------------------------------------------------
// Four bytes per register.  Returns through `code` the raw 2-bit codes (ASCII bits 1..2: A 00, C 01, G 11,
// T 10) of bytes 0..3 in bits 24..31 (byte 0 lowest) and through `flag` 0x80 in every byte that is not one of
// ACGTacgt.  valid <=> (x & 0xD9) == (T-pattern ? 0x50 : 0x41), T-pattern <=> bits(2,1) == (1,0).
__device__ __forceinline__ void classify_word(uint32_t x, uint32_t &code, uint32_t &flag) {
    code = (x & 0x06060606u) * 0x00820820u;
    const uint32_t m = (x >> 2) & ~(x >> 1) & 0x01010101u;           // 1 where the byte has the T pattern
    const uint32_t e = m * 0x0fu + 0x41414141u;                      // expected masked byte: 0x41, or 0x50 for T
    const uint32_t d = (x & 0x59595959u) ^ e;                        // 0 <=> valid (bit 7 is checked below)
    const uint32_t a = d + 0x7f7f7f7fu;                              // bit 7 of each byte <=> byte of d non-zero (d < 0x80)
    flag = (a | x) & 0x80808080u;                                    // bytes >= 0x80 are never DNA
}
// 0x80 in every byte that is 'N' or 'n'
__device__ __forceinline__ uint32_t is_n_word(uint32_t x) {
    const uint32_t d = (x & 0xDFDFDFDFu) ^ 0x4E4E4E4Eu;              // 0 <=> N or n
    return ~((d & 0x7f7f7f7fu) + 0x7f7f7f7fu | d) & 0x80808080u;
}
// gathers bit 7 of the 8 bytes of (w0, w1) into one byte: w0's bytes in bits 0..3, w1's in bits 4..7, returned in bits 24..31
__device__ __forceinline__ uint32_t gather_flags8(uint32_t f0, uint32_t f1) { return (f1 | (f0 >> 4)) * 0x00204081u; }

// 64 flag bytes (16 words of 0x80 marks) -> one 64-bit plane, first byte at bit 63
__device__ __forceinline__ unsigned long long flags_to_plane(const uint32_t (&fb)[16]) {
    uint32_t el[2];
#pragma unroll
    for (int h = 0; h < 2; ++h) {
        uint32_t b[4];
#pragma unroll
        for (int pr = 0; pr < 4; ++pr) b[pr] = gather_flags8(fb[8 * h + 2 * pr], fb[8 * h + 2 * pr + 1]);
        const uint32_t lo2 = __byte_perm(b[0], b[1], 0x0073), hi2 = __byte_perm(b[2], b[3], 0x0073);
        el[h] = __brev(__byte_perm(lo2, hi2, 0x5410));
    }
    return ((unsigned long long)el[0] << 32) | el[1];
}

// 128-bit helpers on (hi, lo) pairs ----------------------------------------------------------------------
__device__ __forceinline__ void shl128(unsigned long long &hi, unsigned long long &lo, int s) {   // s in [0, 128]
    if (s >= 64) { hi = s >= 128 ? 0ull : (lo << (s - 64)); lo = 0ull; }
    else if (s) { hi = (hi << s) | (lo >> (64 - s)); lo <<= s; }
}
// mask of the 128-bit value's bits >= b (b in [0, 128]), as (hi, lo)
__device__ __forceinline__ void mask_ge128(int b, unsigned long long &hi, unsigned long long &lo) {
    if (b >= 64) { lo = 0ull; hi = b >= 128 ? 0ull : (~0ull << (b - 64)); }
    else { hi = ~0ull; lo = ~0ull << b; }
}
__device__ __forceinline__ unsigned long long low_classes(unsigned long long t, int n) {  // lowest n 3-bit classes (n <= 14)
    return t & ((1ull << (3 * n)) - 1ull);
}

// A lane with many flagged bytes (header text, a run of N) gets the whole warp's help: lane j looks at bytes j and
// j + 32 of lane src's 64 bytes, the answers come back by OR-reduction.  Out of line: it runs for a few warps only
// and the sub-tile loop is sensitive to its instruction footprint.
struct HeavyLane { unsigned long long nl, gt, skip, n; };
__device__ __noinline__ HeavyLane heavy_lane_flags(const EncArgs &A, const uint8_t *lut, unsigned long long E, int src,
                                                   int64_t p0, bool full, int lane) {
    constexpr uint32_t FULL = 0xffffffffu;
    const uint32_t Eh = __shfl_sync(FULL, (uint32_t)(E >> 32), src), El = __shfl_sync(FULL, (uint32_t)E, src);
    const int64_t ps = p0 + (int64_t)(src - lane) * LB;          // first byte of that lane
    const uint32_t bit = 0x80000000u >> lane;
    uint32_t w_nl[2] = {0, 0}, w_gt[2] = {0, 0}, w_sk[2] = {0, 0}, w_n[2] = {0, 0};
#pragma unroll
    for (int hh = 0; hh < 2; ++hh) {
        if ((hh ? El : Eh) & bit) {
            const int q = lane + 32 * hh;
            const uint32_t byte = (full || ps + q < A.p_end) ? (uint32_t)__ldg(A.bytes_al + ps + q) : 0u;
            if (byte == '\n') w_nl[hh] = bit;
            if (byte == '>') w_gt[hh] = bit;
            if (lut[byte] == CLS_SKIP) w_sk[hh] = bit;
            if ((byte | 0x20u) == 'n') w_n[hh] = bit;
        }
    }
    HeavyLane r;
    r.nl = ((unsigned long long)__reduce_or_sync(FULL, w_nl[0]) << 32) | __reduce_or_sync(FULL, w_nl[1]);
    r.gt = ((unsigned long long)__reduce_or_sync(FULL, w_gt[0]) << 32) | __reduce_or_sync(FULL, w_gt[1]);
    r.skip = ((unsigned long long)__reduce_or_sync(FULL, w_sk[0]) << 32) | __reduce_or_sync(FULL, w_sk[1]);
    r.n = ((unsigned long long)__reduce_or_sync(FULL, w_n[0]) << 32) | __reduce_or_sync(FULL, w_n[1]);
    return r;
}

// 64-bit plane (first byte at bit 63) of the bytes that are 'N' or 'n'.  Out of line: runs for few warps, and the
// sub-tile loop is sensitive to its instruction footprint.
__device__ __noinline__ unsigned long long n_plane(uint4 v0, uint4 v1, uint4 v2, uint4 v3) {
    const uint32_t xw[16] = {v0.x, v0.y, v0.z, v0.w, v1.x, v1.y, v1.z, v1.w, v2.x, v2.y, v2.z, v2.w, v3.x, v3.y, v3.z, v3.w};
    uint32_t fb[16];
#pragma unroll
    for (int j = 0; j < 16; ++j) fb[j] = is_n_word(xw[j]);
    return flags_to_plane(fb);
}

// Record starts inside the 2 KiB that begin at position lo_pos, for a super-tile with many of them (events r_lo ..
// r_lo + m of rec_offsets): sets their bits in wk[32] (one 64-bit word per lane's bytes), returns how many there are
// and through e_lo the index of the first.  One warp, out of line (rare path).
__device__ __noinline__ int warp_events_many(const EncArgs &A, unsigned long long *wk, int64_t r_lo, int m, int64_t lo_pos,
                                             int lane, int &e_lo) {
    constexpr uint32_t FULL = 0xffffffffu;
    const int64_t hi_pos = lo_pos + WB;
    int lo = 0, hi = m, e_cnt = 0;                               // first event at or after the warp's first byte
    while (lo < hi) {
        const int mid = (lo + hi) >> 1;
        if (rec_pos(A, r_lo + mid) >= lo_pos) hi = mid; else lo = mid + 1;
    }
    e_lo = lo;
    for (int e = lo; e < m; e += 32) {
        const int ee = e + lane;
        const int64_t pp = ee < m ? rec_pos(A, r_lo + ee) : hi_pos;
        const uint32_t inr = __ballot_sync(FULL, pp < hi_pos);
        if (inr && e_cnt == 0) { wk[lane] = 0ull; __syncwarp(); }
        if (pp < hi_pos) atomicOr(&wk[(int)(pp - lo_pos) >> 6], bit_at((int)(pp - lo_pos) & 63));
        e_cnt += __popc(inr);
        if (inr != FULL) break;
    }
    return e_cnt;
}

// ---- scan algebra -----------------------------------------------------------------------------------------
// Agg: a run of consecutive super-tiles seen on its own.  Pre: everything before a point of the byte stream.
struct Agg { uint32_t hasev; int fk, lk, closed, tn; unsigned long long tail; };
struct Pre { int64_t T; QR o; int cnt; unsigned long long tail; };   // tokens of closed records, open record (q, r), tail classes

// earlier run L followed by later run R
__device__ __forceinline__ Agg agg_combine(const Agg &L, const Agg &R, const EncParams &P) {
    Agg G;
    G.hasev = L.hasev | R.hasev;
    G.fk = L.hasev ? L.fk : L.fk + R.fk;
    G.lk = R.hasev ? R.lk : L.lk + R.lk;
    G.closed = L.closed + R.closed + ((L.hasev && R.hasev) ? tok_count32(L.lk + R.fk, P) : 0);
    if (R.hasev || R.tn >= P.k - 1) { G.tn = R.tn; G.tail = R.tail; }
    else {
        const int keepl = min(L.tn, P.k - 1 - R.tn);
        G.tail = (low_classes(L.tail, keepl) << (3 * R.tn)) | R.tail;
        G.tn = R.tn + keepl;
    }
    return G;
}
// prefix X followed by run G
__device__ __forceinline__ Pre pre_extend(const Pre &X, const Agg &G, const EncParams &P) {
    Pre Y;
    if (!G.hasev) {
        Y.T = X.T; Y.o = qr_add(X.o, qr_of((uint32_t)G.fk, P), P.k);
        const int keepx = min(X.cnt, P.k - 1 - G.tn);
        Y.tail = (low_classes(X.tail, keepx) << (3 * G.tn)) | G.tail;
        Y.cnt = keepx + G.tn;
    } else {
        Y.T = X.T + qr_tokens(qr_add(X.o, qr_of((uint32_t)G.fk, P), P.k), P) + G.closed;
        Y.o = qr_of((uint32_t)G.lk, P); Y.tail = G.tail; Y.cnt = G.tn;
    }
    return Y;
}

// ---- emission ---------------------------------------------------------------------------------------
struct SegTab { const int32_t *src, *t, *nwin; };

// One group = R = 16 / sizeof(IdT) consecutive output slots, aligned to 16 bytes in ids_out.  A thread that
// owns a full group inside the window part of one segment reads the stream words once, aligns them with one
// funnel shift per word and cuts R windows at compile-time offsets; everything else goes one token at a time.
template <typename IdT, int K, bool SINGLE, bool REMAP = false>
__device__ __forceinline__ void emit_group_fast(const EncArgs &A, const uint32_t *st, int u, IdT *dst, bool affine) {
    constexpr int R = 16 / (int)sizeof(IdT);
    constexpr int W = 2 * K;                             // code bits per token
    constexpr int CB = W * R;                            // code bits per group
    constexpr int NA = (CB + 31) / 32;
    constexpr int FB = K * R;
    constexpr int NF = (FB + 31) / 32;
    const EncParams &P = A.prm;
    uint32_t a[NA], f[NF];
    {
        const int b = 2 * u, w = b >> 5, s = b & 31;
        uint32_t raw[NA + 1];
#pragma unroll
        for (int i = 0; i <= NA; ++i) raw[i] = st[w + i];
#pragma unroll
        for (int i = 0; i < NA; ++i) a[i] = __funnelshift_l(raw[i + 1], raw[i], s);
    }
    uint32_t anybad = 0;
    {
        const int w = SW_CODE + (u >> 5), s = u & 31;
        uint32_t raw[NF + 1];
#pragma unroll
        for (int i = 0; i <= NF; ++i) raw[i] = st[w + i];
#pragma unroll
        for (int i = 0; i < NF; ++i) {
            f[i] = __funnelshift_l(raw[i + 1], raw[i], s);
            const int lo = i * 32;                       // flag bits [lo, lo + 32) of the group live in f[i]
            anybad |= (lo + 32 <= FB) ? f[i] : (f[i] & ~(0xffffffffu >> (FB - lo)));
        }
    }
    int32_t id[R];
    uint32_t c[R];
#pragma unroll
    for (int t = 0; t < R; ++t) {
        const int bo = W * t, i = bo >> 5, s = bo & 31;
        c[t] = (s + W <= 32) ? ((a[i] >> (32 - s - W)) & ((W == 32) ? 0xffffffffu : ((1u << W) - 1u)))
                             : (__funnelshift_l(a[(i + 1 < NA) ? i + 1 : i], a[i], s) >> (32 - W));
        if (SINGLE) id[t] = affine ? P.nt_ids[0] + (int32_t)c[t] : P.nt_ids[c[t]];
        else id[t] = (REMAP && P.remap4) ? __ldg(P.remap4 + c[t]) : P.base_id + (int32_t)c[t];
    }
    if (anybad) {
#pragma unroll
        for (int t = 0; t < R; ++t) {
            const int bo = K * t, i = bo >> 5, s = bo & 31;
            const uint32_t m = (s + K <= 32) ? ((f[i] >> (32 - s - K)) & ((1u << K) - 1u))
                                             : (__funnelshift_l(f[(i + 1 < NF) ? i + 1 : i], f[i], s) >> (32 - K));
            if (m) id[t] = SINGLE ? (c[t] == 2u ? P.nt_ids[4] : P.unk_id) : ((REMAP && P.remap4) ? kmer_table_id(P, c[t], m, K) : P.unk_id);
        }
    }
    if (sizeof(IdT) == 4) {
        *reinterpret_cast<int4 *>(dst) = make_int4(id[0], id[1], id[2], id[3]);
    } else if (sizeof(IdT) == 2) {
        uint32_t p[4];
#pragma unroll
        for (int j = 0; j < 4; ++j) p[j] = ((uint32_t)id[2 * j] & 0xffffu) | ((uint32_t)id[2 * j + 1] << 16);
        *reinterpret_cast<uint4 *>(dst) = make_uint4(p[0], p[1], p[2], p[3]);
    } else {
        uint32_t p[4];
#pragma unroll
        for (int j = 0; j < 4; ++j)
            p[j] = ((uint32_t)id[4 * j] & 0xffu) | (((uint32_t)id[4 * j + 1] & 0xffu) << 8) |
                   (((uint32_t)id[4 * j + 2] & 0xffu) << 16) | ((uint32_t)id[4 * j + 3] << 24);
        *reinterpret_cast<uint4 *>(dst) = make_uint4(p[0], p[1], p[2], p[3]);
    }
}

// token j (super-tile-relative) of segment-table entry i, any k
template <typename IdT>
__device__ __forceinline__ void emit_token_slow(const EncArgs &A, const uint32_t *st, const SegTab &G, int i, int j, int64_t gidx) {
    const EncParams &P = A.prm;
    const int jj = j - G.t[i], nwin = G.nwin[i], src = G.src[i];
    int32_t id;
    if (P.mode != MODE_KMER) {
        const uint32_t c = class_at(st, src + jj);
        id = c <= CLS_N ? P.nt_ids[c] : P.unk_id;
    } else if (jj < nwin) {
        const int u = src + jj * P.k;
        const uint32_t fl = flags_at(st, u, P.k), cd = code_at(st, u, P.k);
        id = P.remap4 ? kmer_table_id_cold(P, cd, fl, P.k) : (fl ? P.unk_id : (int32_t)(P.base_id + cd));
    } else if (P.tail_policy == TAIL_PER_BASE) {
        const uint32_t c = class_at(st, src + nwin * P.k + (jj - nwin));
        id = c <= CLS_N ? (P.remap4 ? P.nt_ids[c] : (int32_t)(P.base_id + P.four_k + c)) : P.unk_id;
    } else {
        id = P.unk_id;
    }
    store_id<IdT>(A, gidx, id);
}

// largest i < nent with t[i] <= j (t is non-decreasing and t[0] <= j)
__device__ __forceinline__ int find_ent(const SegTab &G, int nent, int j) {
    if (nent <= 4) {
        int i = 0;
        for (int e = 1; e < nent; ++e) i = (G.t[e] <= j) ? e : i;
        return i;
    }
    int lo = 0, hi = nent;
    while (hi - lo > 1) {
        const int mid = (lo + hi) >> 1;
        if (G.t[mid] <= j) lo = mid; else hi = mid;
    }
    return lo;
}

// tokens [ja, jb) (super-tile-relative) of the segment table G; `a` = T0 mod R, gbase = T0 - a
template <typename IdT, int KK>
__device__ __forceinline__ void emit_range(const EncArgs &A, const uint32_t *st, const SegTab &G, int ja, int jb, int nent, int a,
                                           int64_t gbase, int cap_rel, bool vec_ok, bool affine) {
    constexpr int R = 16 / (int)sizeof(IdT);
    const EncParams &P = A.prm;
    const int kk = P.mode == MODE_KMER ? P.k : 0;        // 0: single-nt
    const int kstep = P.mode == MODE_KMER ? P.k : 1;
    IdT *idsA = reinterpret_cast<IdT *>(A.ids) + gbase;
    for (int q = (ja + a) / R + (int)threadIdx.x; q * R - a < jb; q += NT) {
        const int j0 = q * R - a;
        const int lo = j0 < ja ? ja : j0, hi = (j0 + R < jb) ? j0 + R : jb;
        int i = find_ent(G, nent, lo);
        const int jj = lo - G.t[i];
        if (vec_ok && hi - lo == R && jj + R <= G.nwin[i] && q * R + R <= cap_rel) {
            const int u = G.src[i] + jj * kstep;
            IdT *dst = idsA + q * R;
            if constexpr (KK == 0) emit_group_fast<IdT, 1, true>(A, st, u, dst, affine);
            else if constexpr (KK > 0) emit_group_fast<IdT, KK, false>(A, st, u, dst, false);
            else switch (kk) {
                case 0: emit_group_fast<IdT, 1, true>(A, st, u, dst, affine); break;
                case 1: emit_group_fast<IdT, 1, false, true>(A, st, u, dst, false); break;
                case 2: emit_group_fast<IdT, 2, false, true>(A, st, u, dst, false); break;
                case 3: emit_group_fast<IdT, 3, false, true>(A, st, u, dst, false); break;
                case 4: emit_group_fast<IdT, 4, false, true>(A, st, u, dst, false); break;
                case 5: emit_group_fast<IdT, 5, false, true>(A, st, u, dst, false); break;
                case 6: emit_group_fast<IdT, 6, false, true>(A, st, u, dst, false); break;
                default: emit_group_fast<IdT, 8, false, true>(A, st, u, dst, false); break;
            }
        } else {
            for (int j = lo; j < hi; ++j) {
                while (i + 1 < nent && G.t[i + 1] <= j) ++i;
                emit_token_slow<IdT>(A, st, G, i, j, gbase + (int64_t)q * R + (j - j0));
            }
        }
    }
}

// fast groups [qa, qb) of one segment: group q holds tokens q * R - a + (0 .. R-1); token t_lo starts at stream position u0
template <typename IdT, int K, bool SINGLE, bool REMAP = false>
__device__ __forceinline__ void emit_fast_groups(const EncArgs &A, const uint32_t *st, int qa, int qb, int u0, int a, int t_lo,
                                                 IdT *idsA, bool affine) {
    constexpr int R = 16 / (int)sizeof(IdT);
    constexpr int KS = SINGLE ? 1 : K;
    for (int q = qa + (int)threadIdx.x; q < qb; q += NT)
        emit_group_fast<IdT, K, SINGLE, REMAP>(A, st, u0 + (q * R - a - t_lo) * KS, idsA + q * R, affine);
}

// all tokens [0, ntok) of a short segment table (at most EVW + 1 entries): per segment, the 16-byte groups that lie
// inside its window part go through the fast path in one tight loop, the few tokens around them one per thread
template <typename IdT, int KK>
__device__ __forceinline__ void emit_segments(const EncArgs &A, const uint32_t *st, const SegTab &G, int nent, int ntok, int a,
                                              int64_t gbase, int cap_rel, bool vec_ok, bool affine) {
    constexpr int R = 16 / (int)sizeof(IdT);
    const EncParams &P = A.prm;
    const int kk = P.mode == MODE_KMER ? P.k : 0;        // 0: single-nt
    IdT *idsA = reinterpret_cast<IdT *>(A.ids) + gbase;
#pragma unroll 1
    for (int i = 0; i < nent; ++i) {
        const int t_lo = G.t[i], t_hi = i + 1 < nent ? G.t[i + 1] : ntok;
        if (t_hi <= t_lo) continue;
        const int u0 = G.src[i], w_hi = min(t_lo + G.nwin[i], t_hi);
        int qa = 0, qb = 0;
        if (vec_ok) {
            qa = (t_lo + a + R - 1) / R;
            qb = min((w_hi + a) / R, cap_rel / R);
        }
        if (qb > qa) {
            if constexpr (KK == 0) emit_fast_groups<IdT, 1, true>(A, st, qa, qb, u0, a, t_lo, idsA, affine);
            else if constexpr (KK > 0) emit_fast_groups<IdT, KK, false>(A, st, qa, qb, u0, a, t_lo, idsA, false);
            else switch (kk) {
                case 0: emit_fast_groups<IdT, 1, true>(A, st, qa, qb, u0, a, t_lo, idsA, affine); break;
                case 1: emit_fast_groups<IdT, 1, false, true>(A, st, qa, qb, u0, a, t_lo, idsA, false); break;
                case 2: emit_fast_groups<IdT, 2, false, true>(A, st, qa, qb, u0, a, t_lo, idsA, false); break;
                case 3: emit_fast_groups<IdT, 3, false, true>(A, st, qa, qb, u0, a, t_lo, idsA, false); break;
                case 4: emit_fast_groups<IdT, 4, false, true>(A, st, qa, qb, u0, a, t_lo, idsA, false); break;
                case 5: emit_fast_groups<IdT, 5, false, true>(A, st, qa, qb, u0, a, t_lo, idsA, false); break;
                case 6: emit_fast_groups<IdT, 6, false, true>(A, st, qa, qb, u0, a, t_lo, idsA, false); break;
                default: emit_fast_groups<IdT, 8, false, true>(A, st, qa, qb, u0, a, t_lo, idsA, false); break;
            }
            const int h1 = min(t_hi, qa * R - a), h2 = max(t_lo, qb * R - a);     // tokens before / after the fast groups
            const int n1 = h1 - t_lo, n2 = t_hi - h2;
            for (int x = (int)threadIdx.x; x < n1 + n2; x += NT) {
                const int j = x < n1 ? t_lo + x : h2 + (x - n1);
                emit_token_slow<IdT>(A, st, G, i, j, gbase + a + j);
            }
        } else {
            for (int j = t_lo + (int)threadIdx.x; j < t_hi; j += NT) emit_token_slow<IdT>(A, st, G, i, j, gbase + a + j);
        }
    }
}

// ---- pre-pass: record range of every super-tile ----------------------------------------------------------
// first_rec[t] = first r in [0, n_rec] with position >= t * S * TB (n_rec + 1 if none); first_rec[n_tiles] = n_rec + 1
__global__ void __launch_bounds__(256) tile_first_rec_kernel(const __grid_constant__ EncArgs A) {
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");   // the encode kernel may start its prologue now
    asm volatile("griddepcontrol.wait;" ::: "memory");
    if (A.run_if && *A.run_if == 0u) return;                           // the regular-layout fast path has done the work
    const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (t > A.n_tiles) return;
    int64_t lo = 0, hi = A.n_rec + 1;
    if (t < A.n_tiles) {
        const int64_t pos = t * A.S * TB;
        while (lo < hi) {
            const int64_t mid = (lo + hi) >> 1;
            if (rec_pos(A, mid) >= pos) hi = mid; else lo = mid + 1;
        }
    } else {
        lo = A.n_rec + 1;
    }
    A.first_rec[t] = lo;
}

__device__ __forceinline__ void prefetch_l2(const EncArgs &A, int64_t b0) {     // one sub-tile starting at position b0
    int64_t sz = A.p_end - b0;
    sz = sz >= TB ? TB : ((sz + 15) & ~(int64_t)15);
    if (sz > 0)
        asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(A.bytes_al + b0), "r"((uint32_t)sz) : "memory");
}

// ---- next-super-tile preparation (one warp): record range, record-start list, entry line state, L2 prefetch ----
__device__ __forceinline__ void prep_super(const EncArgs &A, Smem5 &sm, int par, unsigned long long ticket, int lane,
                                           int64_t pos_first, int64_t pos_last) {
    constexpr uint32_t FULL = 0xffffffffu;
    const unsigned long long rel = ticket - A.ticket_base;
    const int tile_n = rel >= (unsigned long long)A.n_tiles ? A.n_tiles : (int)rel;
    if (tile_n >= A.n_tiles) {
        if (lane == 0) sm.c_tile[par] = A.n_tiles;
        return;
    }
    const int64_t t0n = (int64_t)tile_n * A.S * TB;
    if (lane < 2 && lane < A.S) prefetch_l2(A, t0n + (int64_t)lane * TB);
    int64_t rlo, rhi;
    if (A.first_rec) { rlo = A.first_rec[tile_n]; rhi = A.first_rec[tile_n + 1]; }
    else {
        // small inputs run without the pre-pass launch: lanes 0 and 1 search rec_offsets for this tile and the next one
        int64_t lo = 0, hi = A.n_rec + 1;
        const int64_t tt = (int64_t)tile_n + (lane & 1);
        if (tt < A.n_tiles) {
            const int64_t pos = tt * A.S * TB;
            while (lo < hi) {
                const int64_t mid = (lo + hi) >> 1;
                if (rec_pos(A, mid) >= pos) hi = mid; else lo = mid + 1;
            }
        } else lo = A.n_rec + 1;
        rlo = __shfl_sync(FULL, lo, 0); rhi = __shfl_sync(FULL, lo, 1);
    }
    const int64_t m64 = rhi - rlo;
    const int m = m64 > 0x7fffffff ? 0x7fffffff : (int)m64;
    if (m <= EVW && lane < m) sm.ev_p[par][lane] = (int)(rec_pos(A, rlo + lane) - t0n);
    // entry line state, read off the 128 bytes in front of the super-tile when they settle it
    uint32_t known = LS_UNKNOWN;
    if (!A.prm.strip_headers) known = LS_IN_LINE;
    else if (t0n <= pos_first || t0n >= pos_last) known = LS_LINE_START;      // no record byte on one side: irrelevant
    else if (m > 0 && rec_pos(A, rlo) == t0n) known = LS_LINE_START;          // a record starts right here
    else {
        const uint32_t wv = __ldg(reinterpret_cast<const uint32_t *>(A.bytes_al + t0n - 128) + lane);
        uint32_t nlm = 0, nsk = 0, gtm = 0;                                     // bit i: byte i of this lane's word
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const uint32_t byte = (wv >> (8 * i)) & 255u;
            nlm |= (uint32_t)(byte == '\n') << i;
            gtm |= (uint32_t)(byte == '>') << i;
            nsk |= (uint32_t)(sm.lut[byte] != CLS_SKIP || byte == '>') << i;   // '>' opens a header even if the table skips it
        }
        int pstar = -1;                                                         // window index of the last line start
        const uint32_t nlb = __ballot_sync(FULL, nlm != 0);
        if (nlb) {
            const int L = 31 - __clz(nlb);
            const uint32_t mm = __shfl_sync(FULL, nlm, L);
            pstar = 4 * L + (31 - __clz(mm)) + 1;
        }
        const int64_t rsw = rec_pos(A, rlo - 1) - (t0n - 128);                  // start of the record holding byte t0n - 1
        if (rsw >= 0 && rsw > pstar) pstar = (int)rsw;
        if (pstar >= 0) {
            uint32_t msk = nsk;
            const int lo = pstar - 4 * lane;                                    // this lane's bytes i >= lo count
            if (lo > 0) msk &= lo >= 4 ? 0u : (0xfu << lo);
            const uint32_t nb = __ballot_sync(FULL, msk != 0);
            if (!nb) known = LS_LINE_START;
            else {
                const int L = __ffs(nb) - 1;
                const uint32_t mm = __shfl_sync(FULL, msk, L), gg = __shfl_sync(FULL, gtm, L);
                known = ((gg >> (__ffs(mm) - 1)) & 1u) ? LS_IN_HEADER : LS_IN_LINE;
            }
        }
    }
    if (lane == 0) { sm.c_tile[par] = tile_n; sm.c_m[par] = m; sm.c_rlo[par] = rlo; sm.c_ls[par] = known; }
}

// exclusive block scan of one int per thread (two barriers)
__device__ __forceinline__ int block_exscan5(int v, Smem5 &sm, int &total) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    int inc = v;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) { int t = __shfl_up_sync(0xffffffffu, inc, d); if (lane >= d) inc += t; }
    if (lane == 31) sm.scan_tmp[warp] = inc;
    __syncthreads();
    int woff = 0, tot = 0;
#pragma unroll
    for (int w = 0; w < NW; ++w) { int t = sm.scan_tmp[w]; if (w < warp) woff += t; tot += t; }
    __syncthreads();
    total = tot;
    return woff + inc - v;
}

// ---- look-back (warp 0): everything before super-tile `tile` ---------------------------------------------------
// Windows of 32 predecessors, nearest first.  Lane l of a window holds tile base - l: an aggregate, an inclusive
// prefix, or nothing yet (then the warp polls).  A window with an inclusive prefix at lane f ends the walk: lanes
// < f extend it.  A window of 32 aggregates is folded into the running aggregate of the nearer tiles.
__device__ __forceinline__ Pre look_back(const EncArgs &A, int tile, int lane) {
    constexpr uint32_t FULL = 0xffffffffu;
    const EncParams &P = A.prm;
    const int k = P.k;
    const uint32_t tagA = (A.gen << 2) | ST_AGG, tagI = (A.gen << 2) | ST_INCL;
    Agg G; G.hasev = 0; G.fk = 0; G.lk = 0; G.closed = 0; G.tn = 0; G.tail = 0;     // tiles nearer than the window
    Pre X; X.T = 0; X.o.q = 0; X.o.r = 0; X.cnt = 0; X.tail = 0;
    for (int base = tile - 1; base >= 0; base -= 32) {
        const int j = base - lane;
        uint4 wa = make_uint4(0, 0, 0, 0), wb = wa, w0 = wa, w1 = wa;
        uint32_t st = ST_INCL;                           // tiles before 0 carry the empty inclusive prefix
        int f = 32; bool ok = true;
        for (int spins = 0;; ++spins) {
            if (j >= 0) {
                const TileDesc &Dj = A.descs[j];
                w0 = ld_vol128(&Dj.i0); w1 = ld_vol128(&Dj.i1); wa = ld_vol128(&Dj.a0); wb = ld_vol128(&Dj.a1);
                st = (w0.x == tagI && w1.x == tagI) ? ST_INCL : ((wa.x == tagA && wb.x == tagA) ? ST_AGG : ST_EMPTY);
            }
            const uint32_t ib = __ballot_sync(FULL, st == ST_INCL);
            f = ib ? __ffs(ib) - 1 : 32;                 // nearest tile with an inclusive prefix
            const uint32_t missing = __ballot_sync(FULL, st == ST_EMPTY) & (f < 32 ? ((1u << f) - 1u) : FULL);
            if (!missing) break;
            if (spins > SPIN_LIMIT) { ok = false; break; }
            __nanosleep(40);
        }
        if (!ok) { if (lane == 0) A.status[1] = 1u; return X; }
        // lanes < f hold aggregates (far = high lane)
        const bool in = lane < f;
        const int fk_l = in ? (int)wa.y : 0, lk_l = (int)wa.z, cl_l = (int)(wa.w & 0x7fffffffu);
        const bool ev_l = in && (wa.w >> 31);
        int Ps = fk_l;                                   // kept-before-first-start summed over lanes >= this one
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) { const int t = __shfl_down_sync(FULL, Ps, d); if (lane + d < 32) Ps += t; }
        const uint32_t evmask = __ballot_sync(FULL, ev_l);
        const int P0 = __shfl_sync(FULL, Ps, 0);
        // the window's lanes < f as one aggregate W
        Agg W; W.hasev = evmask != 0; W.closed = 0;
        if (!evmask) { W.fk = P0; W.lk = P0; }
        else {
            const uint32_t higher = lane == 31 ? 0u : (evmask & ~((2u << lane) - 1u));
            const int ep = higher ? __ffs(higher) - 1 : -1;          // next farther tile with a record start
            const int P_ep = __shfl_sync(FULL, Ps, ep < 0 ? 0 : ep), lk_ep = __shfl_sync(FULL, lk_l, ep < 0 ? 0 : ep);
            int t32 = 0;
            if (ev_l) t32 = cl_l + (ep >= 0 ? tok_count32(lk_ep + Ps - P_ep, P) : 0);
            W.closed = __reduce_add_sync(FULL, t32);
            const int e1 = 31 - __clz(evmask), e0 = __ffs(evmask) - 1;
            W.fk = __shfl_sync(FULL, Ps, e1);
            W.lk = __shfl_sync(FULL, lk_l, e0) + P0 - __shfl_sync(FULL, Ps, e0);
        }
        W.tn = 0; W.tail = 0;
        if (P.mode == MODE_KMER && k > 1) {
            const unsigned long long mytail = (unsigned long long)wb.z | ((unsigned long long)((wb.y >> 4) & 0x3ffu) << 32);
            const int mycnt = (int)(wb.y & 15u);
            const int want = min(k - 1, W.lk);
            for (int l = 0; l < f && W.tn < want; ++l) {
                const unsigned long long tl = __shfl_sync(FULL, mytail, l);
                const int cn = min(__shfl_sync(FULL, mycnt, l), want - W.tn);
                W.tail |= low_classes(tl, cn) << (3 * W.tn);
                W.tn += cn;
                if ((evmask >> l) & 1u) break;
            }
        }
        if (f < 32) {
            // the inclusive prefix at lane f (tiles before 0: empty), extended by W, then by the nearer tiles G
            Pre F;
            const int64_t fT = (int64_t)(((uint64_t)w0.z << 32) | w0.y), fq = (int64_t)(((uint64_t)w1.z << 32) | w1.y);
            const unsigned long long ftail = (unsigned long long)w1.w | ((unsigned long long)((w0.w >> 8) & 0x3ffu) << 32);
            F.T = __shfl_sync(FULL, fT, f); F.o.q = __shfl_sync(FULL, fq, f);
            const uint32_t fw = __shfl_sync(FULL, w0.w, f);
            F.o.r = (int32_t)(fw & 15u); F.cnt = (int)((fw >> 4) & 15u);
            F.tail = __shfl_sync(FULL, ftail, f);
            return pre_extend(pre_extend(F, W, P), G, P);
        }
        G = agg_combine(W, G, P);
    }
    return pre_extend(X, G, P);                          // walked back to the very beginning
}

// ======================================================================================================
// KK: the emission variant compiled in -- 0 single-nt, 1..6 / 8 that k, -1 every variant behind a run-time switch
template <typename IdT, int KK>
__global__ void __launch_bounds__(NT, 1024 / NT) encode_tiles_v5(const __grid_constant__ EncArgs A) {
    extern __shared__ __align__(16) uint8_t smem_raw[];
    Smem5 &sm = *reinterpret_cast<Smem5 *>(smem_raw);
    constexpr uint32_t FULL = 0xffffffffu;
    constexpr int R = 16 / (int)sizeof(IdT);
    const EncParams &P = A.prm;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const uint32_t gen = A.gen;
    const int k = P.k;
    const int S = A.S;
    const int64_t TBS = (int64_t)S * TB;
    const int64_t pos_first = rec_pos(A, 0), pos_last = rec_pos(A, A.n_rec);   // bytes outside are in no record
    const bool affine = P.nt_ids[1] == P.nt_ids[0] + 1 && P.nt_ids[2] == P.nt_ids[0] + 2 && P.nt_ids[3] == P.nt_ids[0] + 3;
    const bool vec_ok = (reinterpret_cast<uintptr_t>(A.ids) & 15) == 0 &&
                        (P.mode != MODE_KMER || (k >= 1 && k <= 6) || k == 8);

    if (tid < 256) sm.lut[tid] = A.lut[tid];
    // launched with programmatic stream serialisation: everything above overlaps the tail of the pre-pass kernel, whose
    // outputs (first_rec, out_offsets) are read only behind this point (a no-op in an ordinary launch)
    asm volatile("griddepcontrol.wait;" ::: "memory");
    if (A.run_if && *A.run_if == 0u) {
        // the regular-layout fast path (encode_fasta.cuh) has encoded this input: only the ticket counter is kept in step
        if (blockIdx.x == 0 && tid == 0) atomicAdd(A.ticket, (unsigned long long)A.n_tiles + gridDim.x);
        return;
    }
    // this launch redoes an input whose layout check failed: tell the host (status word 2, read without synchronising at its
    // next call), which then leaves the regular-layout encoder out for a while
    if (A.run_if && blockIdx.x == 0 && tid == 0) A.status[2] = 1u;
    __syncthreads();
    unsigned long long next_ticket = 0;
    if (warp == NW - 1) {
        if (lane == 0) next_ticket = atomicAdd(A.ticket, 1ull);
        next_ticket = __shfl_sync(FULL, next_ticket, 0);
        prep_super(A, sm, 0, next_ticket, lane, pos_first, pos_last);
    }
    __syncthreads();

    // super-tile A: looped over, aggregate published, waiting for its look-back and emission (stream buffer b ^ 1)
    bool haveA = false;
    int tileA = 0, mA = 0, ktotA = 0;
    int64_t rloA = 0;
    int b = 0;                                                 // stream buffer of super-tile B
#pragma unroll 1
    for (int it = 0;; ++it) {
        const int par = it & 1;
        const int tile = sm.c_tile[par];
        const bool haveB = tile < A.n_tiles;
        if (!haveA && !haveB) break;
        const int m = sm.c_m[par];                             // record starts inside super-tile B
        const int64_t r_lo = sm.c_rlo[par];
        const int64_t t0 = (int64_t)tile * TBS;
        uint32_t *const stB = sm.strm[b];
        int ktot = 0;

        if (haveB) {
            // sub-tiles that hold bytes or the position p_end (where the closing record offset may sit)
            const int64_t rem_b = A.p_end - t0;
            const int S_eff = rem_b >= TBS ? S : (int)(rem_b / TB) + 1;
            const uint32_t ls_known = sm.c_ls[par];
            if (tid == (NW - 1) * 32) next_ticket = atomicAdd(A.ticket, 1ull);
            uint32_t ls_entry = ls_known == LS_UNKNOWN ? LS_IN_LINE : ls_known;
#pragma unroll 1
            for (int pass = 0;; ++pass) {
                // zero the stream (partial words are OR-ed in)
                {
                    const int nb = PEND + S_eff * TB;
                    const int c4 = ((nb >> 4) + 9 + 3) >> 2, f4 = ((nb >> 5) + 10 + 3) >> 2;
                    uint4 *s4 = reinterpret_cast<uint4 *>(stB);
                    for (int i = tid; i < c4; i += NT) s4[i] = make_uint4(0, 0, 0, 0);
                    for (int i = tid; i < f4; i += NT) s4[SW_CODE / 4 + i] = make_uint4(0, 0, 0, 0);
                }
                int base = 0;                                        // kept bases of the sub-tiles done so far
                uint32_t ls_use = ls_entry;                          // entry line state of the sub-tile
                uint32_t t_hr = 0, t_x = LS_LINE_START;              // line-state summary of the super-tile (thread NT-1)
#pragma unroll 1
                for (int s = 0; s < S_eff; ++s) {
                    const int sp = s & 1;
                    const int64_t ts0 = t0 + (int64_t)s * TB;
                    const int64_t p0 = ts0 + (int64_t)tid * LB;          // position of this thread's first byte
                    const bool full = ts0 + TB <= A.p_end;
                    // ================= P1: load, classify, exceptions, line-state summary ==========================
                    uint4 v[4];
                    {
                        const uint4 *src = reinterpret_cast<const uint4 *>(A.bytes_al + p0);
                        if (full) {
#pragma unroll
                            for (int j = 0; j < 4; ++j) v[j] = __ldg(src + j);
                        } else {
#pragma unroll
                            for (int j = 0; j < 4; ++j) v[j] = (p0 + 16 * j < A.p_end) ? __ldg(src + j) : make_uint4(0, 0, 0, 0);
                        }
                    }
                    if (tid == 0 && s + 2 < S_eff) prefetch_l2(A, ts0 + 2 * TB);
                    // record starts inside this warp's 2 KiB: events [e_lo, e_lo + e_cnt) of the super-tile
                    int e_lo = 0, e_cnt = 0;
                    unsigned long long rs = 0ull;
                    const int wb = s * TB + warp * WB;                   // super-tile position of the warp's first byte
                    if (m > 0) {
                        if (m <= EVW) {
                            const int p = lane < m ? sm.ev_p[par][lane] - wb : -1;
                            const uint32_t inr = __ballot_sync(FULL, (unsigned)p < (unsigned)WB);
                            if (inr) {
                                e_lo = __ffs(inr) - 1; e_cnt = __popc(inr);
                                sm.wk[warp][lane] = 0ull;
                                __syncwarp();
                                if ((inr >> lane) & 1u) atomicOr(&sm.wk[warp][p >> 6], bit_at(p & 63));
                                __syncwarp();
                                rs = sm.wk[warp][lane];
                            }
                        } else {
                            e_cnt = warp_events_many(A, sm.wk[warp], r_lo, m, t0 + wb, lane, e_lo);
                            if (e_cnt) { __syncwarp(); rs = sm.wk[warp][lane]; }
                        }
                    }
                    unsigned long long chi, clo, bad, E;                 // code plane (128 b), not-ACGT plane, exception plane
                    {
                        const uint32_t *xw = reinterpret_cast<const uint32_t *>(v);
                        uint32_t cb[16], fb[16];
#pragma unroll
                        for (int j = 0; j < 16; ++j) classify_word(xw[j], cb[j], fb[j]);
                        uint32_t C[4];
#pragma unroll
                        for (int h = 0; h < 4; ++h) {
                            // top bytes of four products -> one LSB-first word of 16 bases -> MSB first, Gray -> binary
                            const uint32_t lo2 = __byte_perm(cb[4 * h], cb[4 * h + 1], 0x0073);
                            const uint32_t hi2 = __byte_perm(cb[4 * h + 2], cb[4 * h + 3], 0x0073);
                            const uint32_t y = __brev(__byte_perm(lo2, hi2, 0x5410));
                            C[h] = ((y & 0x55555555u) << 1) | (((y >> 1) ^ y) & 0x55555555u);
                        }
                        chi = ((unsigned long long)C[0] << 32) | C[1];
                        clo = ((unsigned long long)C[2] << 32) | C[3];
                        uint32_t anyf = 0;
#pragma unroll
                        for (int j = 0; j < 16; ++j) anyf |= fb[j];
                        E = anyf ? flags_to_plane(fb) : 0ull;
                        if (!P.fast_lut) E = ~0ull;
                        bad = E;
                        // runs of N: classified arithmetically too (their digit is already 2), not one LUT trip per byte
                        // (lanes that are still heavy afterwards -- header text -- are handled by the whole warp below)
                        if (P.fast_lut && P.fast_n && __any_sync(FULL, __popcll(E) >= 4)) {
                            E &= ~n_plane(v[0], v[1], v[2], v[3]);
                        }
                    }
                    unsigned long long skip = 0, nl = 0, gt = 0;
                    bool coop_done = false;
                    if (P.fast_lut) {
                        uint32_t hv = __ballot_sync(FULL, __popcll(E) >= 4);
                        while (hv) {
                            const int src = __ffs(hv) - 1;
                            hv &= hv - 1;
                            const HeavyLane hl = heavy_lane_flags(A, sm.lut, E, src, p0, full, lane);
                            if (lane == src) {
                                nl = hl.nl; gt = hl.gt; skip = hl.skip;
                                // 'N' / 'n' already carry digit 2 and stay flagged in `bad`: no second trip for them
                                if (P.fast_n) E &= ~hl.n;
                                coop_done = true;
                            }
                        }
                    }
                    {
                        const uint8_t *vb = A.bytes_al + p0;
                        unsigned long long rem = coop_done ? 0ull : E;
                        while (rem) {
                            const int q = __clzll((long long)rem);
                            const unsigned long long bq = bit_at(q);
                            rem ^= bq;
                            const uint32_t byte = (full || p0 + q < A.p_end) ? (uint32_t)__ldg(vb + q) : 0u;
                            // first trip: only what the line state and the keep mask need; the class of a flagged byte
                            // is looked up in P2, and only if the byte is kept (header bytes never are)
                            if (byte == '\n') nl |= bq;
                            if (byte == '>') gt |= bq;
                            if (sm.lut[byte] == CLS_SKIP) skip |= bq;
                        }
                    }
                    // line state: thread summary (has_reset, exit state if the entry state is LINE_START), scanned over the warp
                    const unsigned long long osk = skip & ~nl & ~gt;   // SKIP bytes that neither end nor start a line
                    const unsigned long long ls_base = (nl >> 1) | rs; // line starts: after each '\n' and at each record start
                    auto settle = [&](unsigned long long ls, bool &pending) {   // move line starts over non-newline SKIP bytes
                        pending = (nl & 1ull) != 0;
                        unsigned long long t;
                        while ((t = ls & osk) != 0) { pending = pending || (t & 1ull); ls = (ls & ~t) | (t >> 1); }
                        return ls;
                    };
                    uint32_t e_hr = 0, e_x = LS_LINE_START, s_hr = 0, s_x = LS_LINE_START;
                    if (P.strip_headers && !__any_sync(FULL, (nl | gt | rs | osk) != 0ull)) {
                        // nothing in this warp's 2 KiB touches the line state: every summary is (no reset, IN_LINE)
                        s_x = LS_IN_LINE;
                        if (lane == 31) sm.warp_ls[sp][warp] = LS_IN_LINE;
                        e_x = lane == 0 ? LS_LINE_START : LS_IN_LINE;
                    } else if (P.strip_headers) {
                        if ((gt | osk) == 0ull) {
                            // no '>' and nothing to settle over: after the last byte the line is open unless that byte is '\n'
                            s_x = (nl & 1ull) ? LS_LINE_START : LS_IN_LINE;
                        } else {
                            bool pend0;
                            const unsigned long long ls0 = settle(ls_base | bit_at(0), pend0);
                            if (pend0) s_x = LS_LINE_START;
                            else if (!ls0) s_x = LS_LINE_START;
                            else s_x = (gt & (ls0 & (~ls0 + 1ull))) ? LS_IN_HEADER : LS_IN_LINE;   // lowest set bit = last line start
                        }
                        s_hr = (nl | rs) != 0;
#pragma unroll
                        for (int d = 1; d < 32; d <<= 1) {
                            const uint32_t o_hr = __shfl_up_sync(FULL, s_hr, d), o_x = __shfl_up_sync(FULL, s_x, d);
                            if (lane >= d) {                             // (earlier o) then (later s)
                                s_x = ls_apply(s_hr, s_x, o_x);
                                s_hr |= o_hr;
                            }
                        }
                        if (lane == 31) sm.warp_ls[sp][warp] = (s_hr << 2) | s_x;
                        e_hr = __shfl_up_sync(FULL, s_hr, 1); e_x = __shfl_up_sync(FULL, s_x, 1);
                        if (lane == 0) { e_hr = 0; e_x = LS_LINE_START; }  // identity
                    }
                    __syncthreads();                                     // ---- B: warp line-state summaries (zeroed stream when s == 0)

                    // ================= P2: header mask, keep mask, compaction, warp scan ==============================
                    unsigned long long hdr = 0;
                    if (P.strip_headers) {
                        uint32_t z_hr = 0, z_x = LS_LINE_START;          // summary of the warps before this one
                        {
                            uint32_t wl[NW], w_or = 0u, w_and = ~0u;
#pragma unroll
                            for (int q4 = 0; q4 < NW / 4; ++q4) {
                                const uint4 t4 = *reinterpret_cast<const uint4 *>(&sm.warp_ls[sp][4 * q4]);
                                wl[4 * q4] = t4.x; wl[4 * q4 + 1] = t4.y; wl[4 * q4 + 2] = t4.z; wl[4 * q4 + 3] = t4.w;
                                w_or |= (t4.x | t4.y) | (t4.z | t4.w); w_and &= (t4.x & t4.y) & (t4.z & t4.w);
                            }
                            if (w_or == LS_IN_LINE && w_and == LS_IN_LINE) {     // all (no reset, IN_LINE)
                                if (warp > 0) z_x = LS_IN_LINE;
                            } else {
#pragma unroll
                                for (int w = 0; w < NW - 1; ++w) {
                                    const uint32_t g_hr = wl[w] >> 2, g_x = wl[w] & 3u;
                                    if (w < warp) { z_x = ls_apply(g_hr, g_x, z_x); z_hr |= g_hr; }
                                }
                            }
                        }
                        uint32_t st_in = ls_apply(z_hr, z_x, ls_use);
                        if (tid == NT - 1) {                             // whole sub-tile: exit state, super-tile summary
                            z_x = ls_apply(s_hr, s_x, z_x); z_hr |= s_hr;
                            sm.ls_sub[sp] = ls_apply(z_hr, z_x, ls_use);
                            t_x = ls_apply(z_hr, z_x, t_x); t_hr |= z_hr;
                        }
                        st_in = ls_apply(e_hr, e_x, st_in);
                        if ((nl | gt | rs) == 0ull) {                    // no line ends or starts here: all header or none
                            if (st_in == LS_IN_HEADER) hdr = ~0ull;
                        } else if (gt == 0ull && st_in != LS_IN_HEADER) {
                            // no '>' here and not inside a header: nothing of this thread's bytes is header
                        } else {
                        bool pd;
                        const unsigned long long ls = settle(ls_base | (st_in == LS_LINE_START ? bit_at(0) : 0ull), pd);
                        unsigned long long hs = ls & gt;                 // header lines that start inside this thread's bytes
                        if (st_in == LS_IN_HEADER) {
                            const int a = first_pos(nl), bb = first_pos(rs);
                            const int e = (bb <= a) ? bb - 1 : a;        // through the '\n', or up to a record start
                            if (e >= 0) hdr |= (e >= 63) ? ~0ull : ~from_pos(e + 1);
                        }
                        while (hs) {
                            const int h = __clzll((long long)hs);
                            hs &= ~bit_at(h);
                            const int a = first_pos(nl & from_pos(h)), bb = first_pos(rs & from_pos(h + 1));
                            const int e = (bb <= a) ? bb - 1 : a;
                            hdr |= from_pos(h) & ((e >= 63) ? ~0ull : ~from_pos(e + 1));
                        }
                        }
                    }
                    unsigned long long keep = ~skip & ~hdr;
                    if (p0 < pos_first || p0 + LB > pos_last) {
                        const int64_t a = pos_first - p0, bb = pos_last - p0;       // in-record positions are [a, bb)
                        const unsigned long long ma = a <= 0 ? ~0ull : from_pos((int)(a > 64 ? 64 : a));
                        const unsigned long long mb = bb <= 0 ? 0ull : (bb >= 64 ? ~0ull : ~from_pos((int)bb));
                        keep &= ma & mb;
                    }
                    {
                        // second trip through the LUT: class of every kept byte the arithmetic did not prove to be ACGT
                        const uint8_t *vb = A.bytes_al + p0;
                        unsigned long long rem = E & keep;
                        while (rem) {
                            const int q = __clzll((long long)rem);
                            const unsigned long long bq = bit_at(q);
                            rem ^= bq;
                            const uint32_t byte = (full || p0 + q < A.p_end) ? (uint32_t)__ldg(vb + q) : 0u;
                            const uint32_t c = sm.lut[byte];
                            if (c < CLS_N) bad &= ~bq;
                            const unsigned long long cc = c < CLS_N ? c : (c == CLS_N ? 2u : 1u);
                            const int sh = 62 - 2 * (q & 31);
                            if (q < 32) chi = (chi & ~(3ull << sh)) | (cc << sh);
                            else clo = (clo & ~(3ull << sh)) | (cc << sh);
                        }
                    }
                    const bool wfull = __all_sync(FULL, keep == ~0ull);  // nothing dropped in this warp's 2 KiB
                    const int n = __popcll(keep);
                    if (n == 0) { chi = clo = bad = 0ull; }
                    else if (n == 63) {
                        // one dropped byte (the newline of a wrapped FASTA line): its flag bit and its two code bits go
                        const int lo = __ffsll((long long)~keep) - 1;                      // plane bit of the dropped byte
                        const unsigned long long lm = (1ull << lo) - 1ull;
                        bad = (bad & ~(lm | (1ull << lo))) | ((bad & lm) << 1);
                        if (lo >= 32) {
                            const int pb = 2 * lo - 64;                                    // its code bits: chi bits pb, pb + 1
                            const unsigned long long up = pb + 2 < 64 ? (~0ull << (pb + 2)) : 0ull;
                            chi = (chi & up) | ((chi & ((1ull << pb) - 1ull)) << 2) | (clo >> 62);
                            clo <<= 2;
                        } else {
                            const int pb = 2 * lo;                                         // clo bits pb, pb + 1
                            const unsigned long long up = pb + 2 < 64 ? (~0ull << (pb + 2)) : 0ull;
                            clo = (clo & up) | ((clo & ((1ull << pb) - 1ull)) << 2);
                        }
                    } else if (n != 64) {
                        // delete the dropped runs from the planes, last run first so earlier positions stay valid
                        unsigned long long drop = ~keep;
                        while (drop) {
                            const int lo = __ffsll((long long)drop) - 1;                   // lowest bit of the last run
                            const unsigned long long t = ~(drop >> lo);
                            const int len = t ? __ffsll((long long)t) - 1 : 64 - lo;       // run length (bits lo .. lo+len-1)
                            const unsigned long long lm = (1ull << lo) - 1ull;             // bits below the run
                            const unsigned long long hm = (lo + len >= 64) ? 0ull : (~0ull << (lo + len));
                            drop &= hm;
                            bad = (bad & hm) | ((bad & lm) << len);
                            unsigned long long mh, ml, kh, kl;
                            mask_ge128(2 * (lo + len), mh, ml);                            // code bits above the run stay
                            kh = chi & mh; kl = clo & ml;
                            unsigned long long lh, ll;                                     // code bits below the run move up
                            mask_ge128(2 * lo, lh, ll);
                            unsigned long long bh = chi & ~lh, bl = clo & ~ll;
                            shl128(bh, bl, 2 * len);
                            chi = kh | bh; clo = kl | bl;
                        }
                    }
                    int inc = n;
                    if (wfull) inc = LB * (lane + 1);
                    else {
#pragma unroll
                        for (int d = 1; d < 32; d <<= 1) { const int t = __shfl_up_sync(FULL, inc, d); if (lane >= d) inc += t; }
                    }
                    if (lane == 31) sm.warp_cnt[sp][warp] = inc;
                    __syncthreads();                                     // ---- C: warp counts, sub-tile exit line state

                    // ================= P3: stream append; kept-base index of the record starts =========================
                    int woff = 0, ksub = 0;
{
                        int wc[NW];
#pragma unroll
                        for (int q4 = 0; q4 < NW / 4; ++q4) {
                            const int4 t4 = *reinterpret_cast<const int4 *>(&sm.warp_cnt[sp][4 * q4]);
                            wc[4 * q4] = t4.x; wc[4 * q4 + 1] = t4.y; wc[4 * q4 + 2] = t4.z; wc[4 * q4 + 3] = t4.w;
                        }
#pragma unroll
                        for (int w = 0; w < NW; ++w) { woff += (w < warp) ? wc[w] : 0; ksub += wc[w]; }
                    }
                    if (wfull) {
                        // every lane appends 64 bases: whole words, the bits shared with the lane before come by shuffle
                        const int u = PEND + base + woff + LB * lane;
                        const uint32_t C0 = (uint32_t)(chi >> 32), C1 = (uint32_t)chi, C2 = (uint32_t)(clo >> 32), C3 = (uint32_t)clo;
                        const uint32_t bh = (uint32_t)(bad >> 32), bl = (uint32_t)bad;
                        uint32_t pC3 = __shfl_up_sync(FULL, C3, 1), pbl = __shfl_up_sync(FULL, bl, 1);
                        if (lane == 0) { pC3 = 0u; pbl = 0u; }
                        const int cw0 = u >> 4, csh = 2 * (u & 15);      // csh, fsh are the same in every lane
                        const uint32_t c0 = __funnelshift_r(C0, pC3, csh);
                        if (lane == 0) { if (c0) atomicOr(&stB[cw0], c0); } else stB[cw0] = c0;
                        stB[cw0 + 1] = __funnelshift_r(C1, C0, csh);
                        stB[cw0 + 2] = __funnelshift_r(C2, C1, csh);
                        stB[cw0 + 3] = __funnelshift_r(C3, C2, csh);
                        const int fw0 = SW_CODE + (u >> 5), fsh = u & 31;
                        const uint32_t f0 = __funnelshift_r(bh, pbl, fsh);
                        if (lane == 0) { if (f0) atomicOr(&stB[fw0], f0); } else stB[fw0] = f0;
                        stB[fw0 + 1] = __funnelshift_r(bl, bh, fsh);
                        if (lane == 31) {
                            const uint32_t c4 = __funnelshift_r(0u, C3, csh), f2 = __funnelshift_r(0u, bl, fsh);
                            if (csh && c4) atomicOr(&stB[cw0 + 4], c4);
                            if (fsh && f2) atomicOr(&stB[fw0 + 2], f2);
                        }
                    } else if (n > 0) {
                        const int u = PEND + base + woff + inc - n;      // stream position of this thread's first kept base
                        const uint32_t C0 = (uint32_t)(chi >> 32), C1 = (uint32_t)chi, C2 = (uint32_t)(clo >> 32), C3 = (uint32_t)clo;
                        const int cw0 = u >> 4, csh = 2 * (u & 15);
                        const int cend = csh + 2 * n;                    // code bits [csh, cend) of the words from cw0 on
                        uint32_t cwv[5];
                        cwv[0] = C0 >> csh;
                        cwv[1] = __funnelshift_r(C1, C0, csh);
                        cwv[2] = __funnelshift_r(C2, C1, csh);
                        cwv[3] = __funnelshift_r(C3, C2, csh);
                        cwv[4] = __funnelshift_r(0u, C3, csh);
#pragma unroll
                        for (int i = 0; i < 5; ++i) {
                            if (32 * i < cend) {
                                const bool whole = (i > 0 || csh == 0) && 32 * (i + 1) <= cend;
                                if (whole) stB[cw0 + i] = cwv[i];
                                else if (cwv[i]) atomicOr(&stB[cw0 + i], cwv[i]);
                            }
                        }
                        const uint32_t bh = (uint32_t)(bad >> 32), bl = (uint32_t)bad;
                        const int fw0 = SW_CODE + (u >> 5), fsh = u & 31, fend = fsh + n;
                        uint32_t bwv[3];
                        bwv[0] = bh >> fsh; bwv[1] = __funnelshift_r(bl, bh, fsh); bwv[2] = __funnelshift_r(0u, bl, fsh);
#pragma unroll
                        for (int i = 0; i < 3; ++i) {
                            if (32 * i < fend) {
                                const bool whole = (i > 0 || fsh == 0) && 32 * (i + 1) <= fend;
                                if (whole) stB[fw0 + i] = bwv[i];
                                else if (bwv[i]) atomicOr(&stB[fw0 + i], bwv[i]);
                            }
                        }
                    }
                    if (e_cnt) {                                         // warp-uniform
                        sm.wk[warp][lane] = keep; sm.offw[warp][lane] = (uint16_t)(inc - n);
                        __syncwarp();
                        for (int e = e_lo + lane; e < e_lo + e_cnt; e += 32) {
                            const int p = (m <= EVW ? sm.ev_p[par][e] : (int)(rec_pos(A, r_lo + e) - t0)) - wb;
                            const int o = p >> 6, q = p & 63;
                            const int kidx = base + woff + (int)sm.offw[warp][o] + (q ? __popcll(sm.wk[warp][o] >> (64 - q)) : 0);
                            if (m <= EVW) sm.ev_k[b][e] = kidx; else A.rec_k[r_lo + e] = kidx;
                        }
                        __syncwarp();
                    }
                    base += ksub;
                    if (P.strip_headers) ls_use = sm.ls_sub[sp];
                }
                ktot = base;
                if (P.strip_headers && tid == NT - 1) sm.t_ls = (t_hr << 2) | t_x;
                if (ls_known != LS_UNKNOWN || pass == 1) break;
                __syncthreads();                                         // ---- summary of the super-tile
                // ---- warp 0: entry line state of the super-tile from the chain ------------------------------------
                if (warp == 0) {
                    uint32_t state = LS_LINE_START;
                    const uint32_t tagL = gen << 8;
                    const uint32_t tl = sm.t_ls, u_hr = tl >> 2, u_x = tl & 3u;
                    if (lane == 0) st_vol32(&A.ls[tile], tagL | ((u_hr ? LK_FINAL : LK_SUMMARY) << 2) | u_x);
                    bool ok = true;
                    uint32_t carry = LS_LINE_START; bool have_carry = false;
                    for (int bs = tile - 1;; bs -= 32) {                 // tile > 0: tile 0's entry state is always known
                        const int j = bs - lane;
                        uint32_t kind = LK_FINAL, val = LS_LINE_START;     // tiles before 0: known LINE_START
                        int f = 32;
                        for (int spins = 0;; ++spins) {
                            if (j >= 0) {
                                const uint32_t a = ld_vol32(&A.ls[j]);
                                kind = (a >> 8) == (gen & 0xffffffu) ? ((a >> 2) & 3u) : LK_NONE;
                                val = a & 3u;
                            }
                            const uint32_t tb = __ballot_sync(FULL, kind == LK_FINAL);
                            f = tb ? __ffs(tb) - 1 : 32;                   // nearest tile whose exit state is final
                            const uint32_t missing = __ballot_sync(FULL, kind == LK_NONE) & (f < 32 ? ((1u << f) - 1u) : FULL);
                            if (!missing) break;
                            if (spins > SPIN_LIMIT) { ok = false; break; }
                            __nanosleep(40);
                        }
                        if (!ok) break;
                        // the value that survives is the farthest non-LINE_START one at or before the final tile
                        const uint32_t nb = __ballot_sync(FULL, val != LS_LINE_START && lane <= f);
                        if (nb) { carry = __shfl_sync(FULL, val, 31 - __clz(nb)); have_carry = true; }
                        if (f < 32) break;
                    }
                    state = have_carry ? carry : LS_LINE_START;
                    if (!ok && lane == 0) A.status[1] = 1u;
                    if (lane == 0) {
                        st_vol32(&A.ls[tile], tagL | (LK_FINAL << 2) | ls_apply(u_hr, u_x, state));
                        sm.ls_in = state; sm.redo = state != LS_IN_LINE;
                    }
                }
                __syncthreads();                                         // ---- entry line state
                if (!sm.redo) break;
                ls_entry = sm.ls_in;
            }
        }
        __syncthreads();                                             // ---- D: stream B, record-start indices, summary

        // ================= warp NW-1: next ticket; warp 1: aggregate(B); warp 0: look-back(A) ======================
        if (warp == NW - 1) {
            if (haveB) {
                next_ticket = __shfl_sync(FULL, next_ticket, 0);
                prep_super(A, sm, par ^ 1, next_ticket, lane, pos_first, pos_last);
            } else if (lane == 0) {
                sm.c_tile[par ^ 1] = A.n_tiles;
            }
        }
        // the three one-warp jobs run side by side: warp NW-1 prepares the next super-tile, warp 1 publishes the aggregate
        // of B, warp 0 looks back for A
        const uint32_t tagA = (gen << 2) | ST_AGG, tagI = (gen << 2) | ST_INCL;
        if (warp == 1 || warp == 0) {
            if (warp == 1 && haveB) {
                // ---- aggregate of super-tile B and the segment table of its record starts --------------------------
                int fk, lk, closed = 0, ntok = 0;
                if (m == 0) { fk = ktot; lk = ktot; }
                else if (m <= EVW) {
                    const int ke = lane < m ? sm.ev_k[b][lane] : ktot;
                    int kn = __shfl_down_sync(FULL, ke, 1);
                    if (lane >= m - 1) kn = ktot;
                    const int ne = kn - ke;
                    const int nw = (int)div_k((uint32_t)ne, P);
                    // records that close inside emit windows + tail; the one still open at the end only windows
                    const int te = lane < m - 1 ? nw + tail_tokens(ne - nw * k, P) : (lane == m - 1 ? nw : 0);
                    int ti = te;
#pragma unroll
                    for (int d = 1; d < 32; d <<= 1) { const int t = __shfl_up_sync(FULL, ti, d); if (lane >= d) ti += t; }
                    const int ex = ti - te;
                    ntok = __shfl_sync(FULL, ti, 31); closed = __shfl_sync(FULL, ex, m - 1);
                    if (lane < m) { sm.seg_src[b][1 + lane] = PEND + ke; sm.seg_t[b][1 + lane] = ex; sm.seg_nwin[b][1 + lane] = nw; }
                    fk = __shfl_sync(FULL, ke, 0); lk = __shfl_sync(FULL, ne, m - 1);
                } else {
                    // many record starts: only the aggregate here, the table is built chunk by chunk at emission
                    fk = 0;
                    for (int c0 = 0; c0 < m; c0 += 32) {
                        const int e = c0 + lane;
                        const int ke = e < m ? __ldcg(A.rec_k + r_lo + e) : ktot;
                        int kn = __shfl_down_sync(FULL, ke, 1);
                        if (lane == 31) kn = e + 1 < m ? __ldcg(A.rec_k + r_lo + e + 1) : ktot;
                        const int te = e < m - 1 ? tok_count32(kn - ke, P) : 0;
                        closed += __reduce_add_sync(FULL, te);
                        if (c0 == 0) fk = __shfl_sync(FULL, ke, 0);
                    }
                    lk = ktot - __ldcg(A.rec_k + r_lo + m - 1);
                }
                // last tn = min(k - 1, lk) classes of the super-tile, 3 bits each, newest lowest
                const int tn = min(k - 1, lk);
                unsigned long long gtail = 0;
                {
                    unsigned long long tl = 0;
                    if (lane < tn) tl = (unsigned long long)class_at(stB, PEND + ktot - tn + lane) << (3 * (tn - 1 - lane));
                    gtail = ((unsigned long long)__reduce_or_sync(FULL, (uint32_t)(tl >> 32)) << 32) | __reduce_or_sync(FULL, (uint32_t)tl);
                }
                if (lane == 0) {
                    TileDesc &D = A.descs[tile];
                    st_vol128(&D.a0, make_uint4(tagA, (uint32_t)fk, (uint32_t)lk, (uint32_t)closed | ((uint32_t)(m > 0) << 31)));
                    st_vol128(&D.a1, make_uint4(tagA, (uint32_t)tn | ((uint32_t)(gtail >> 32) << 4), (uint32_t)gtail, 0u));
                    TileAgg &g = sm.ag[b];
                    g.fk = fk; g.lk = lk; g.closed = closed; g.tn = tn; g.ntok = ntok; g.hasev = m > 0; g.tail = gtail;
                    // line-state word of a super-tile whose entry state was known up front
                    if (P.strip_headers && sm.c_ls[par] != LS_UNKNOWN) {
                        const uint32_t tl = sm.t_ls;
                        st_vol32(&A.ls[tile], (gen << 8) | (LK_FINAL << 2) | ls_apply(tl >> 2, tl & 3u, sm.c_ls[par]));
                    }
                }
            }
            if (warp == 0 && haveA) {
                // ---- look-back for super-tile A, its inclusive prefix, its segment-table entry 0 ---------------------
                const int ba = b ^ 1;
                uint32_t *const stA = sm.strm[ba];
                const Pre X = look_back(A, tileA, lane);
                Agg g;
                {
                    const TileAgg &t = sm.ag[ba];
                    g.hasev = t.hasev; g.fk = t.fk; g.lk = t.lk; g.closed = t.closed; g.tn = t.tn; g.tail = t.tail;
                }
                const int pend = P.mode == MODE_KMER ? X.o.r : 0;
                const int nbase0 = pend + g.fk;
                const int nwin0 = (int)div_k((uint32_t)nbase0, P), rem0 = nbase0 - nwin0 * k;
                const int tok0 = nwin0 + (g.hasev ? tail_tokens(rem0, P) : 0);
                const Pre Y = pre_extend(X, g, P);
                if (lane == 0) {
                    TileDesc &D = A.descs[tileA];
                    st_vol128(&D.i0, make_uint4(tagI, (uint32_t)Y.T, (uint32_t)((uint64_t)Y.T >> 32),
                                                (uint32_t)Y.o.r | ((uint32_t)Y.cnt << 4) | ((uint32_t)(Y.tail >> 32) << 8)));
                    st_vol128(&D.i1, make_uint4(tagI, (uint32_t)Y.o.q, (uint32_t)((uint64_t)Y.o.q >> 32), (uint32_t)Y.tail));
                }
                // carried bases of the open record go in front of the stream
                {
                    uint32_t cw = 0, fw = 0;
                    if (lane < pend) {
                        const uint32_t c = (uint32_t)(X.tail >> (3 * (pend - 1 - lane))) & 7u;
                        const int uu = PEND - pend + lane;
                        const uint32_t dg = c < CLS_N ? c : (c == CLS_N ? 2u : 1u);
                        cw = dg << (30 - 2 * uu);
                        fw = c >= CLS_N ? (1u << (31 - uu)) : 0u;
                    }
                    cw = __reduce_or_sync(FULL, cw); fw = __reduce_or_sync(FULL, fw);
                    if (lane == 0) { stA[0] = cw; if (fw) atomicOr(&stA[SW_CODE], fw); }
                }
                if (mA <= EVW && lane < mA) sm.seg_t[ba][1 + lane] += tok0;
                if (lane == 0) {
                    sm.seg_src[ba][0] = PEND - pend; sm.seg_t[ba][0] = 0; sm.seg_nwin[ba][0] = nwin0;
                    sm.tok0 = tok0; sm.ntok = sm.ag[ba].ntok + tok0;
                    sm.T0 = A.out_bias + X.T + X.o.q;
                }
            }
        }
        __syncthreads();                                         // ---- E: prefix of A known, next super-tile prepared

        // ================= emit super-tile A ========================================================================
        if (haveA) {
            const int ba = b ^ 1;
            const uint32_t *const stA = sm.strm[ba];
            const int64_t T0 = sm.T0;
            const int a = (int)(T0 & (R - 1));
            const int64_t gbase = T0 - a;
            const int64_t capl = A.ids_cap - gbase;
            const int cap_rel = capl < 0 ? 0 : (capl > 0x7fffffff ? 0x7fffffff : (int)capl);
            const int tok0 = sm.tok0;
            if (mA <= EVW) {
                SegTab G; G.src = sm.seg_src[ba]; G.t = sm.seg_t[ba]; G.nwin = sm.seg_nwin[ba];
                if (tid < mA) A.out_off[rloA + tid] = T0 + G.t[1 + tid];
                emit_segments<IdT, KK>(A, stA, G, mA + 1, sm.ntok, a, gbase, cap_rel, vec_ok, affine);
            } else {
                SegTab G; G.src = sm.ent_src; G.t = sm.ent_t; G.nwin = sm.ent_nwin;
                if (tid == 0) { sm.ent_src[0] = sm.seg_src[ba][0]; sm.ent_t[0] = 0; sm.ent_nwin[0] = sm.seg_nwin[ba][0]; }
                int tbase = tok0;                                // super-tile-relative token index of the chunk's first record
                for (int c0 = 0; c0 < mA; c0 += NT) {
                    const int cm = min(NT, mA - c0), e = c0 + tid;
                    int ke = ktotA, ne = 0, te = 0, nw = 0;
                    if (e < mA) {
                        ke = __ldcg(A.rec_k + rloA + e);
                        const int kn = e + 1 < mA ? __ldcg(A.rec_k + rloA + e + 1) : ktotA;
                        ne = kn - ke;
                        nw = (int)div_k((uint32_t)ne, P);
                        te = e + 1 < mA ? nw + tail_tokens(ne - nw * k, P) : nw;
                    }
                    int total;
                    const int ex = block_exscan5(te, sm, total);
                    if (e < mA) {
                        sm.ent_src[1 + tid] = PEND + ke; sm.ent_t[1 + tid] = tbase + ex; sm.ent_nwin[1 + tid] = nw;
                        A.out_off[rloA + e] = T0 + tbase + ex;
                    }
                    if (c0 > 0 && tid == 0) { sm.ent_src[0] = 0; sm.ent_t[0] = tbase; sm.ent_nwin[0] = 0; }
                    __syncthreads();
                    emit_range<IdT, KK>(A, stA, G, c0 == 0 ? 0 : tbase, tbase + total, cm + 1, a, gbase, cap_rel, vec_ok, affine);
                    tbase += total;
                    __syncthreads();
                }
            }
        }
        __syncthreads();                                         // ---- A's buffer and tables are free again
        haveA = haveB; tileA = tile; mA = m; rloA = r_lo; ktotA = ktot; b ^= 1;
    }
}

}  // namespace v5
}  // namespace dtk
