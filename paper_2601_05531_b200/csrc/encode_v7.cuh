// encode_v7.cuh -- single-pass classify + strip + {single-nt | k-mer} + CSR offsets: eight compute warps with private
// regions and one scan warp per CTA, no block barrier inside the byte loop.
//
// A persistent CTA (288 threads, 3 per SM) claims flat TILES of S x 16 KiB input bytes in order (atomic ticket).
// Inside a tile each of the eight COMPUTE warps owns one contiguous REGION of S x 2 KiB and walks it in steps of
// 2 KiB (64 contiguous bytes per lane, four 16-byte loads straight into registers):
//   classify ("256-entry LUT"; Alg. 1): ACGT in either case is recognised arithmetically on
//     four bytes per 32-bit register and gathered into per-lane bit planes (2-bit base-4 digits, MSB first, and a
//     "not ACGT" flag plane); every byte the arithmetic does not prove to be ACGT goes through the 256-entry LUT in
//     shared memory -- the table stays the specification.  The lane's raw bytes are staged in a private, swizzled
//     shared-memory slot so a flagged byte is read back with one LDS instead of a second global load.
//   strip: newline / header / SKIP bytes are deleted from the planes in registers; line state is a warp-uniform value
//     carried along the region (a warp whose 2 KiB hold no '>', no record start and no odd SKIP byte never scans it).
//   append: the kept bases go to the region's own slice of the tile's kept-base stream in shared memory (warp prefix
//     by ballot + popc; even lanes store, odd lanes read-modify-write, so no shared-memory atomics on the fast path).
// The SCAN warp (warp 8) does everything that is serial, one tile ahead or behind the compute warps, so they never
// wait for it: ticket + record range + L2 prefetch of the next tile; per-tile aggregate (kept bases before the first /
// after the last record start, tokens of records closed inside, the last k-1 classes) published for the chained scan;
// decoupled look-back with walk-back over windows of 32 predecessors; the tile's segment table (one entry per record
// start and per region start); out_offsets of the records that start in the tile; the 15-base halo behind each region.
// Hand-offs are named barriers (bar.arrive / bar.sync): PREP (scan -> compute), DONE (compute -> scan), READY
// (scan -> compute).  Emission: every compute warp cuts the tokens whose first base lies in its own region from the
// stream in groups of 16 output bytes (one funnel-shift alignment per group, windows at compile-time offsets, one
// 16-byte store straight to ids_out).
// DENSE mode (create-time spec with no SKIP class and strip_headers = 0, SURVEY.md section 7 hard part 2): kept bases
// = bytes, so every position is closed-form from rec_offsets -- no chain, no look-back, no compaction; out_offsets
// come from a scan over the record lengths in the pre-pass.
// Input bytes are read from HBM exactly once and ids written exactly once.
#pragma once
#include "common.cuh"

namespace dtk {
namespace v7 {

constexpr int NWC = NT / 32;                 // compute warps
static_assert(NWC == 8, "eight regions per tile");
constexpr int NT7 = NT + 32;                 // + the scan warp
constexpr int WB = 32 * LB;                  // input bytes per warp per step (2 KiB)
constexpr int REG_CAP = S_MAX * WB;          // kept bases one region can hold
constexpr int REG_STRIDE = REG_CAP + 128;    // stream slots between region starts: halo + both planes stay 16-byte aligned
constexpr int PEND = 128;                    // stream slots in front of region 0 (carried bases sit in the last 15)
constexpr int HALO = 15;                     // kept bases copied behind each region (k - 1 at most)
constexpr int STREAM_BASES = PEND + NWC * REG_STRIDE;
constexpr int SW_CODE = ((STREAM_BASES / 16 + 8) + 3) & ~3;
constexpr int SW_FLAG = ((STREAM_BASES / 32 + 8) + 3) & ~3;
constexpr int SW_ALL = SW_CODE + SW_FLAG;    // multiple of 4 words
constexpr int EV_MAX = 64;                   // record starts per tile handled through the shared-memory tables
constexpr int NSE = EV_MAX + NWC;            // segment-table entries: entry 0, the record starts, 7 region starts
constexpr uint32_t LS_UNKNOWN = 3;
enum : int { BAR_PREP = 1, BAR_READY = 3 };   // PREP alternates between ids 1 and 2, READY between 3 and 4; DONE is a polled counter

struct TileAgg {                             // aggregate of one tile, kept until its look-back
    int32_t fk, lk, closed, tn;              // kept before first / after last record start, tokens of records inside, tail classes held
    uint32_t hasev;
    unsigned long long tail;                 // last tn classes, 3 bits each, newest lowest
};

struct TileCtl {                             // scan warp -> compute warps, one per loop iteration (double-buffered)
    int32_t tile;                            // tile to compact (-1: none)
    int32_t buf;                             // its stream / table buffer
    int32_t emit;                            // after the compaction: emit the tile held in buffer emit_buf
    int32_t emit_buf;
    int32_t emit_generic;                    // that tile has more record starts than the tables hold
    int32_t last;                            // leave the loop after this iteration
};

struct TileBuf {                             // per stream buffer
    long long rlo;                           // first record starting inside the tile (index into rec_offsets)
    long long T0;                            // global index of the tile's first token
    int32_t tile, m;                         // m: record starts inside (clipped to int); written by the preparation
    long long e_rlo;                         // copies for the emission (the preparation of the tile after next may
    int32_t e_tile, e_m;                     //   already be rewriting tile / m / rlo / ev_p while this tile is emitted)
    int32_t ktot, ntok;                      // kept bases, tokens
    int32_t pend, tok0, nwin0;               // entry 0: carried bases, its tokens, its windows
    int32_t cum[NWC + 1];                    // kept bases before each region
    int32_t rbase[NWC];                      // stream slot of each region's first kept base (reg_slot + what was dropped)
    int32_t reg_cnt[NWC];
    int32_t reg_hfix[NWC];                   // kept bases in front of the region's first line reset (dropped if the
                                             //   region turns out to have started inside a header line)
    uint32_t reg_ls[NWC];                    // known << 8 | entry << 4 | hr << 2 | x   (region line-state record)
    int32_t reg_e0[NWC + 1];                 // segment-table range of each region
    uint16_t ev_p[EV_MAX];                   // tile positions of the record starts
    int32_t ev_k[EV_MAX];                    // kept bases in front of each: region-relative | region << 16, then logical
    int32_t le_src[EV_MAX + 1], le_t[EV_MAX + 2], le_nwin[EV_MAX + 1];   // logical entries: 0 = open record, 1 + e = record start e
    int32_t se_src[NSE], se_t[NSE + 1], se_nwin[NSE];                    // split at region starts, physical stream positions
    TileAgg ag;
};

struct Smem7 {
    uint32_t strm[2][SW_ALL];                // per buffer -- code stream: slot u at word u>>4, bits 31-2(u&15), 30-2(u&15);
                                             // flag stream at + SW_CODE: slot u at word u>>5, bit 31-(u&31)
    uint4 stage[NWC][128];                   // per compute warp: the lanes' raw 64 bytes
    unsigned long long wk[NWC][32];          // per compute warp: record-start bitmap, then keep masks (event steps only)
    uint16_t offw[NWC][32];
    TileBuf tb[2];
    TileCtl ctl[2];
    int32_t done_cnt;                        // regions compacted since the kernel started (compute warps -> scan warp)
    uint8_t lut[256];
};
static_assert(sizeof(Smem7) <= 76288, "three CTAs per SM (227 KiB, 1 KiB reserved per CTA)");

// ---------------------------------------------------------------------------------------- small helpers
__device__ __forceinline__ void bar_sync(int id) { asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(NT7) : "memory"); }
__device__ __forceinline__ void bar_arrive(int id) { asm volatile("bar.arrive %0, %1;" ::"r"(id), "r"(NT7) : "memory"); }

__device__ __forceinline__ unsigned long long bit_at(int q) { return 0x8000000000000000ull >> q; }          // q in 0..63
__device__ __forceinline__ unsigned long long from_pos(int q) { return q >= 64 ? 0ull : (~0ull >> q); }   // positions >= q
__device__ __forceinline__ int first_pos(unsigned long long m) { return m ? __clzll((long long)m) : 64; }

__device__ __forceinline__ int reg_slot(int w) { return PEND + w * REG_STRIDE; }   // stream slot of region w's first base

// k digits starting at slot u (k <= 16) of the stream buffer st
__device__ __forceinline__ uint32_t code_at(const uint32_t *st, int u, int k) {
    const int b = 2 * u, w = b >> 5, s = b & 31;
    return __funnelshift_l(st[w + 1], st[w], s) >> (32 - 2 * k);
}
__device__ __forceinline__ uint32_t flags_at(const uint32_t *st, int u, int k) {    // k flag bits starting at slot u
    const int w = u >> 5, s = u & 31;
    const uint32_t *f = st + SW_CODE;
    return __funnelshift_l(f[w + 1], f[w], s) >> (32 - k);
}
// class code 0..5 of slot u: ACGT from the code plane; flagged bases carry digit 2 for N (what the arithmetic
// classification yields for 'N' / 'n') and digit 1 for UNK
__device__ __forceinline__ uint32_t class_at(const uint32_t *st, int u) {
    const uint32_t c = code_at(st, u, 1);
    return flags_at(st, u, 1) ? (c == 2u ? CLS_N : CLS_UNK) : c;
}
// stream slot of logical kept-base index u of the tile (u < 0: carried bases in front of region 0)
__device__ __forceinline__ int slot_of(const TileBuf &tb, int u) {
    int r = 0;
#pragma unroll
    for (int w = 1; w < NWC; ++w) r += (u >= tb.cum[w]) ? 1 : 0;
    return tb.rbase[r] + (u - tb.cum[r]);
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

// 64 bytes -> code plane C[0..3] (16 bases per word, first base in bits 31..30, binary digits A C G T = 0 1 2 3) and
// the plane E of bytes that are not ACGTacgt (first byte at bit 63)
__device__ __forceinline__ void classify64(const uint4 (&v)[4], uint32_t (&C)[4], unsigned long long &E) {
    const uint32_t *xw = reinterpret_cast<const uint32_t *>(v);
    uint32_t cb[16], fb[16];
#pragma unroll
    for (int j = 0; j < 16; ++j) classify_word(xw[j], cb[j], fb[j]);
#pragma unroll
    for (int h = 0; h < 4; ++h) {
        // top bytes of four products -> one LSB-first word of 16 bases -> MSB first, Gray -> binary
        const uint32_t lo2 = __byte_perm(cb[4 * h], cb[4 * h + 1], 0x0073);
        const uint32_t hi2 = __byte_perm(cb[4 * h + 2], cb[4 * h + 3], 0x0073);
        const uint32_t y = __brev(__byte_perm(lo2, hi2, 0x5410));
        C[h] = ((y & 0x55555555u) << 1) | (((y >> 1) ^ y) & 0x55555555u);
    }
    uint32_t anyf = 0;
#pragma unroll
    for (int j = 0; j < 16; ++j) anyf |= fb[j];
    E = anyf ? flags_to_plane(fb) : 0ull;
}

// 64-bit plane (first byte at bit 63) of the bytes that are 'N' or 'n'.  Out of line: runs for few warps.
__device__ __noinline__ unsigned long long n_plane(uint4 v0, uint4 v1, uint4 v2, uint4 v3) {
    const uint32_t xw[16] = {v0.x, v0.y, v0.z, v0.w, v1.x, v1.y, v1.z, v1.w, v2.x, v2.y, v2.z, v2.w, v3.x, v3.y, v3.z, v3.w};
    uint32_t fb[16];
#pragma unroll
    for (int j = 0; j < 16; ++j) fb[j] = is_n_word(xw[j]);
    return flags_to_plane(fb);
}

// 128-bit helpers on (hi, lo) pairs ----------------------------------------------------------------------
__device__ __forceinline__ void shl128(unsigned long long &hi, unsigned long long &lo, int s) {   // s in [0, 128]
    if (s >= 64) { hi = s >= 128 ? 0ull : (lo << (s - 64)); lo = 0ull; }
    else if (s) { hi = (hi << s) | (lo >> (64 - s)); lo <<= s; }
}
__device__ __forceinline__ void mask_ge128(int b, unsigned long long &hi, unsigned long long &lo) {  // bits >= b
    if (b >= 64) { lo = 0ull; hi = b >= 128 ? 0ull : (~0ull << (b - 64)); }
    else { hi = ~0ull; lo = ~0ull << b; }
}
__device__ __forceinline__ unsigned long long low_classes(unsigned long long t, int n) {  // lowest n 3-bit classes (n <= 14)
    return t & ((1ull << (3 * n)) - 1ull);
}

// base q (0..63 from the front) leaves the planes: later bases move up one slot, a zero slot enters at the end
__device__ __forceinline__ void delete_one(uint32_t (&C)[4], unsigned long long &bad, int q) {
    const int q2 = 2 * q;
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        const uint32_t nx = j < 3 ? C[j + 1] : 0u;
        const uint32_t S = __funnelshift_l(nx, C[j], 2);                       // the word one base further on
        const uint32_t T = __funnelshift_rc(0xffffffffu, 0u, max(q2 - 32 * j, 0));   // slots >= q of this word
        C[j] = (C[j] & ~T) | (S & T);
    }
    const unsigned long long T = from_pos(q);
    bad = (bad & ~T) | ((bad << 1) & T);
}
// every dropped run leaves the planes (last run first so earlier positions stay valid).  Out of line: header and
// record-boundary lanes only.
__device__ __noinline__ void delete_runs(uint32_t (&C)[4], unsigned long long &bad, unsigned long long keep) {
    unsigned long long chi = ((unsigned long long)C[0] << 32) | C[1], clo = ((unsigned long long)C[2] << 32) | C[3];
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
    C[0] = (uint32_t)(chi >> 32); C[1] = (uint32_t)chi; C[2] = (uint32_t)(clo >> 32); C[3] = (uint32_t)clo;
}
__device__ __forceinline__ void set_digit(uint32_t (&C)[4], int q, uint32_t d) {
    const int sh = 30 - 2 * (q & 15);
#pragma unroll
    for (int j = 0; j < 4; ++j)
        if ((q >> 4) == j) C[j] = (C[j] & ~(3u << sh)) | (d << sh);
}

// ---- scan algebra -----------------------------------------------------------------------------------------
// Agg: a run of consecutive tiles seen on its own.  Pre: everything before a point of the byte stream.
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
// One group = R = 16 / sizeof(IdT) consecutive output slots, aligned to 16 bytes in ids_out.  A lane that owns a
// full group inside the window part of one segment reads the stream words once, aligns them with one funnel shift
// per word and cuts R windows at compile-time offsets; everything else goes one token at a time.
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

// token jj (entry-relative) of a segment-table entry (src = stream slot of its first base, nwin windows, then tail
// tokens), any k
template <typename IdT>
__device__ __forceinline__ void emit_token_slow(const EncArgs &A, const uint32_t *st, int src, int nwin, int jj, int64_t gidx) {
    const EncParams &P = A.prm;
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

// fast groups [qa, qb) of one segment, 32 lanes: group q holds tokens q * R - a + (0 .. R-1); token t_lo starts at slot u0
template <typename IdT, int K, bool SINGLE, bool REMAP = false>
__device__ __forceinline__ void emit_fast_groups(const EncArgs &A, const uint32_t *st, int qa, int qb, int u0, int a, int t_lo,
                                                 IdT *idsA, bool affine, int lane) {
    constexpr int R = 16 / (int)sizeof(IdT);
    constexpr int KS = SINGLE ? 1 : K;
    for (int q = qa + lane; q < qb; q += 32)
        emit_group_fast<IdT, K, SINGLE, REMAP>(A, st, u0 + (q * R - a - t_lo) * KS, idsA + q * R, affine);
}

// one compute warp emits the tokens whose first base lies in its region: per segment-table entry, the 16-byte groups
// that lie inside its window part go through the fast path in one tight loop, the few tokens around them one per lane
template <typename IdT, int KK>
__device__ __forceinline__ void emit_region(const EncArgs &A, const uint32_t *st, const TileBuf &tb, int w, int lane,
                                            bool vec_ok, bool affine) {
    constexpr int R = 16 / (int)sizeof(IdT);
    const EncParams &P = A.prm;
    const int kk = P.mode == MODE_KMER ? P.k : 0;        // 0: single-nt
    const int64_t T0 = tb.T0;
    const int a = (int)(T0 & (R - 1));
    const int64_t gbase = T0 - a;
    const int64_t capl = A.ids_cap - gbase;
    const int cap_rel = capl < 0 ? 0 : (capl > 0x7fffffff ? 0x7fffffff : (int)capl);
    IdT *idsA = reinterpret_cast<IdT *>(A.ids) + gbase;
    const int e1 = tb.reg_e0[w + 1];
#pragma unroll 1
    for (int i = tb.reg_e0[w]; i < e1; ++i) {
        const int t_lo = tb.se_t[i], t_hi = tb.se_t[i + 1];
        if (t_hi <= t_lo) continue;
        const int u0 = tb.se_src[i], nwin = tb.se_nwin[i], w_hi = min(t_lo + nwin, t_hi);
        int qa = 0, qb = 0;
        if (vec_ok) {
            qa = (t_lo + a + R - 1) / R;
            qb = min((w_hi + a) / R, cap_rel / R);
        }
        if (qb > qa) {
            if constexpr (KK == 0) emit_fast_groups<IdT, 1, true>(A, st, qa, qb, u0, a, t_lo, idsA, affine, lane);
            else if constexpr (KK > 0) emit_fast_groups<IdT, KK, false>(A, st, qa, qb, u0, a, t_lo, idsA, false, lane);
            else switch (kk) {
                case 0: emit_fast_groups<IdT, 1, true>(A, st, qa, qb, u0, a, t_lo, idsA, affine, lane); break;
                case 1: emit_fast_groups<IdT, 1, false, true>(A, st, qa, qb, u0, a, t_lo, idsA, false, lane); break;
                case 2: emit_fast_groups<IdT, 2, false, true>(A, st, qa, qb, u0, a, t_lo, idsA, false, lane); break;
                case 3: emit_fast_groups<IdT, 3, false, true>(A, st, qa, qb, u0, a, t_lo, idsA, false, lane); break;
                case 4: emit_fast_groups<IdT, 4, false, true>(A, st, qa, qb, u0, a, t_lo, idsA, false, lane); break;
                case 5: emit_fast_groups<IdT, 5, false, true>(A, st, qa, qb, u0, a, t_lo, idsA, false, lane); break;
                case 6: emit_fast_groups<IdT, 6, false, true>(A, st, qa, qb, u0, a, t_lo, idsA, false, lane); break;
                default: emit_fast_groups<IdT, 8, false, true>(A, st, qa, qb, u0, a, t_lo, idsA, false, lane); break;
            }
            const int h1 = min(t_hi, qa * R - a), h2 = max(t_lo, qb * R - a);     // tokens before / after the fast groups
            const int n1 = h1 - t_lo, n2 = t_hi - h2;
            for (int x = lane; x < n1 + n2; x += 32) {
                const int j = x < n1 ? t_lo + x : h2 + (x - n1);
                emit_token_slow<IdT>(A, st, u0, nwin, j - t_lo, gbase + a + j);
            }
        } else {
            for (int j = t_lo + lane; j < t_hi; j += 32) emit_token_slow<IdT>(A, st, u0, nwin, j - t_lo, gbase + a + j);
        }
    }
}

// ---- pre-pass ---------------------------------------------------------------------------------------------
// first_rec[t] = first r in [0, n_rec] with position >= t * S * TB (n_rec + 1 if none); first_rec[n_tiles] = n_rec + 1
__device__ __forceinline__ void prefetch_l2(const EncArgs &A, int64_t b0, int bytes) {   // [b0, b0 + bytes) clipped to the input
    int64_t sz = A.p_end - b0;
    sz = sz >= bytes ? bytes : ((sz + 15) & ~(int64_t)15);
    if (sz > 0)
        asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(A.bytes_al + b0), "r"((uint32_t)sz) : "memory");
}

// DENSE mode pre-pass: out_offsets = exclusive scan of the per-record token counts, which follow from the record
// lengths alone (kept bases = bytes).  Chained scan over blocks of 2048 records; the chain words reuse the tile
// descriptor array (a0 of descriptor b: { tag, status, sum lo, sum hi }).
constexpr int DS_NT = 256, DS_PER = 8, DS_BLK = DS_NT * DS_PER;
__device__ __forceinline__ int64_t dense_tokens(int64_t len, const EncParams &P) {
    if (P.mode != MODE_KMER) return len;
    const int64_t q = len / P.k;
    return q + tail_tokens((int)(len - q * P.k), P);
}
// One launch: blocks [0, nb_first) write first_rec (256 tiles each), the blocks behind them run the offsets scan.
__global__ void __launch_bounds__(DS_NT) dense_prepass_kernel(const __grid_constant__ EncArgs A, TileDesc *chain, int nb_first) {
    __shared__ long long wsum[DS_NT / 32];
    __shared__ long long s_base;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");   // the encode kernel may start its prologue now
    if ((int)blockIdx.x < nb_first) {
        const int64_t t = (int64_t)blockIdx.x * DS_NT + tid;
        if (t > A.n_tiles) return;
        int64_t lo = 0, hi = A.n_rec + 1;
        if (t < A.n_tiles) {
            const int64_t pos = t * A.S * TB;
            while (lo < hi) {
                const int64_t mid = (lo + hi) >> 1;
                if (rec_pos(A, mid) >= pos) hi = mid; else lo = mid + 1;
            }
        } else lo = A.n_rec + 1;
        A.first_rec[t] = lo;
        return;
    }
    const int b = (int)blockIdx.x - nb_first;
    const int64_t r0 = (int64_t)b * DS_BLK + (int64_t)tid * DS_PER;
    long long v[DS_PER], run = 0;
#pragma unroll
    for (int i = 0; i < DS_PER; ++i) {
        const int64_t r = r0 + i;
        v[i] = r < A.n_rec ? dense_tokens(A.rec_off[r + 1] - A.rec_off[r], A.prm) : 0;
        run += v[i];
    }
    long long inc = run;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) { const long long t = __shfl_up_sync(0xffffffffu, inc, d); if (lane >= d) inc += t; }
    if (lane == 31) wsum[warp] = inc;
    __syncthreads();
    long long woff = 0, tot = 0;
#pragma unroll
    for (int w = 0; w < DS_NT / 32; ++w) { const long long t = wsum[w]; if (w < warp) woff += t; tot += t; }
    const uint32_t tagA = (A.gen << 2) | ST_AGG, tagI = (A.gen << 2) | ST_INCL;
    if (tid == 0) {
        long long base = 0;
        if (b > 0) {
            st_vol128(&chain[b].a0, make_uint4(tagA, 0u, (uint32_t)tot, (uint32_t)((unsigned long long)tot >> 32)));
            for (int j = b - 1; j >= 0; --j) {
                uint4 w;
                int spins = 0;
                for (;;) {
                    w = ld_vol128(&chain[j].a0);
                    if (w.x == tagA || w.x == tagI) break;
                    if (++spins > SPIN_LIMIT) { A.status[1] = 1u; break; }
                    __nanosleep(20);
                }
                base += (long long)(((unsigned long long)w.w << 32) | w.z);
                if (w.x == tagI) break;
            }
        }
        const long long incl = base + tot;
        st_vol128(&chain[b].a0, make_uint4(tagI, 0u, (uint32_t)incl, (uint32_t)((unsigned long long)incl >> 32)));
        s_base = base;
        if ((int64_t)(b + 1) * DS_BLK >= A.n_rec) A.out_off[A.n_rec] = A.out_bias + incl;
    }
    __syncthreads();
    long long ex = s_base + woff + inc - run + A.out_bias;
#pragma unroll
    for (int i = 0; i < DS_PER; ++i) {
        const int64_t r = r0 + i;
        if (r < A.n_rec) A.out_off[r] = ex;
        ex += v[i];
    }
}

// ---- look-back (scan warp): everything before tile `tile` -------------------------------------------------------
// Two levels.  Tiles form groups of 32; the scan warp of a group's last tile publishes the GROUP aggregate (all 32
// tile aggregates folded) as soon as it has seen them, and that tile's inclusive prefix is the group's inclusive
// prefix.  A look-back is then: one window over the predecessors inside the tile's own group, and windows of 32
// GROUPS (1024 tiles each) from there on -- two reads in practice, however many tiles are in flight.
// Lane l of a window holds item base - l: an aggregate, an inclusive prefix, or nothing yet.  A window with an
// inclusive prefix at lane f ends the walk: lanes < f extend it.  A window of aggregates only is folded into the
// running aggregate of the nearer items.  ONE attempt: when a needed item has published nothing yet, `ready` comes
// back false and the caller tries again later (the scan warp never blocks here).
struct Win { uint4 a0, a1, i0, i1; uint32_t st; };

// lanes < f of a window (aggregates; far = high lane) folded into one aggregate
__device__ __forceinline__ Agg fold_window(const Win &w, int f, const EncParams &P, int lane) {
    constexpr uint32_t FULL = 0xffffffffu;
    const int k = P.k;
    const bool in = lane < f;
    const int fk_l = in ? (int)w.a0.y : 0, lk_l = (int)w.a0.z, cl_l = (int)(w.a0.w & 0x7fffffffu);
    const bool ev_l = in && (w.a0.w >> 31);
    int Ps = fk_l;                                       // kept-before-first-start summed over lanes >= this one
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) { const int t = __shfl_down_sync(FULL, Ps, d); if (lane + d < 32) Ps += t; }
    const uint32_t evmask = __ballot_sync(FULL, ev_l);
    const int P0 = __shfl_sync(FULL, Ps, 0);
    Agg W; W.hasev = evmask != 0; W.closed = 0;
    if (!evmask) { W.fk = P0; W.lk = P0; }
    else {
        const uint32_t higher = lane == 31 ? 0u : (evmask & ~((2u << lane) - 1u));
        const int ep = higher ? __ffs(higher) - 1 : -1;              // next farther item with a record start
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
        const unsigned long long mytail = (unsigned long long)w.a1.z | ((unsigned long long)((w.a1.y >> 4) & 0x3ffu) << 32);
        const int mycnt = (int)(w.a1.y & 15u);
        const int want = min(k - 1, W.lk);
        for (int l = 0; l < f && W.tn < want; ++l) {
            const unsigned long long tl = __shfl_sync(FULL, mytail, l);
            const int cn = min(__shfl_sync(FULL, mycnt, l), want - W.tn);
            W.tail |= low_classes(tl, cn) << (3 * W.tn);
            W.tn += cn;
            if ((evmask >> l) & 1u) break;
        }
    }
    return W;
}
// the inclusive prefix held by lane f of a window
__device__ __forceinline__ Pre incl_at(const Win &w, int f) {
    constexpr uint32_t FULL = 0xffffffffu;
    Pre F;
    const int64_t fT = (int64_t)(((uint64_t)w.i0.z << 32) | w.i0.y), fq = (int64_t)(((uint64_t)w.i1.z << 32) | w.i1.y);
    const unsigned long long ftail = (unsigned long long)w.i1.w | ((unsigned long long)((w.i0.w >> 8) & 0x3ffu) << 32);
    F.T = __shfl_sync(FULL, fT, f); F.o.q = __shfl_sync(FULL, fq, f);
    const uint32_t fw = __shfl_sync(FULL, w.i0.w, f);
    F.o.r = (int32_t)(fw & 15u); F.cnt = (int)((fw >> 4) & 15u);
    F.tail = __shfl_sync(FULL, ftail, f);
    return F;
}
__device__ __forceinline__ void publish_agg(TileDesc *D, uint32_t tagA, const Agg &g) {
    st_vol128(&D->a0, make_uint4(tagA, (uint32_t)g.fk, (uint32_t)g.lk, (uint32_t)g.closed | ((uint32_t)(g.hasev != 0) << 31)));
    st_vol128(&D->a1, make_uint4(tagA, (uint32_t)g.tn | ((uint32_t)(g.tail >> 32) << 4), (uint32_t)g.tail, 0u));
}

// own: the tile's own aggregate (the last tile of a group folds it into the group aggregate it publishes)
__device__ __noinline__ Pre look_back(const EncArgs &A, int tile, const Agg &own, int lane, bool force, bool &ready) {
    constexpr uint32_t FULL = 0xffffffffu;
    const EncParams &P = A.prm;
    const uint32_t tagA = (A.gen << 2) | ST_AGG, tagI = (A.gen << 2) | ST_INCL;
    Agg G; G.hasev = 0; G.fk = 0; G.lk = 0; G.closed = 0; G.tn = 0; G.tail = 0;     // items nearer than the window
    Pre X; X.T = 0; X.o.q = 0; X.o.r = 0; X.cnt = 0; X.tail = 0;
    ready = true;
    const int p = tile & 31, grp = tile >> 5;
    Win w;
    // ---- level 0: the predecessors inside the tile's own group (lane l <-> tile - 1 - l, l < p) ------------------
    if (p > 0) {
        w.a0 = w.a1 = w.i0 = w.i1 = make_uint4(0, 0, 0, 0);
        w.st = ST_AGG;                                   // lanes >= p: not part of this window
        if (lane < p) {
            const TileDesc &Dj = A.descs[tile - 1 - lane];
            w.i0 = ld_vol128(&Dj.i0); w.i1 = ld_vol128(&Dj.i1); w.a0 = ld_vol128(&Dj.a0); w.a1 = ld_vol128(&Dj.a1);
            w.st = (w.i0.x == tagI && w.i1.x == tagI) ? ST_INCL : ((w.a0.x == tagA && w.a1.x == tagA) ? ST_AGG : ST_EMPTY);
        }
        const uint32_t ib = __ballot_sync(FULL, w.st == ST_INCL);
        const int f = ib ? __ffs(ib) - 1 : p;            // nearest tile with an inclusive prefix
        const uint32_t empty = __ballot_sync(FULL, w.st == ST_EMPTY);
        if (p == 31) {
            // last tile of its group: the group aggregate goes out as soon as all 32 tile aggregates are there
            const uint32_t noagg = __ballot_sync(FULL, lane < 31 && !(w.a0.x == tagA && w.a1.x == tagA));
            if (noagg) { ready = force; return X; }
            const Agg Wall = fold_window(w, 31, P, lane);
            const Agg GG = agg_combine(Wall, own, P);
            if (lane == 0) publish_agg(&A.gdescs[grp], tagA, GG);
        }
        if (empty & ((1u << f) - 1u)) { ready = force; return X; }      // (forced: the chain is broken, the status word says so)
        const Agg W = fold_window(w, f, P, lane);
        if (ib) return pre_extend(incl_at(w, f), W, P);
        G = W;
    }
    // ---- level 1: whole groups (lane l <-> group base - l): group aggregate, or the inclusive prefix of its last tile
    for (int base = grp - 1; base >= 0; base -= 32) {
        const int j = base - lane;
        w.a0 = w.a1 = w.i0 = w.i1 = make_uint4(0, 0, 0, 0);
        w.st = ST_INCL;                                  // groups before 0 carry the empty inclusive prefix
        if (j >= 0) {
            const TileDesc &Dt = A.descs[32 * j + 31];
            const TileDesc &Dg = A.gdescs[j];
            w.i0 = ld_vol128(&Dt.i0); w.i1 = ld_vol128(&Dt.i1); w.a0 = ld_vol128(&Dg.a0); w.a1 = ld_vol128(&Dg.a1);
            w.st = (w.i0.x == tagI && w.i1.x == tagI) ? ST_INCL : ((w.a0.x == tagA && w.a1.x == tagA) ? ST_AGG : ST_EMPTY);
        }
        const uint32_t ib = __ballot_sync(FULL, w.st == ST_INCL);
        const int f = ib ? __ffs(ib) - 1 : 32;
        const uint32_t missing = __ballot_sync(FULL, w.st == ST_EMPTY) & (f < 32 ? ((1u << f) - 1u) : FULL);
        if (missing) { ready = force; return X; }
        const Agg W = fold_window(w, f, P, lane);
        if (f < 32) {
            Pre F = incl_at(w, f);
            if (base - f < 0) { F = X; }                 // walked past group 0: the empty prefix
            return pre_extend(pre_extend(F, W, P), G, P);
        }
        G = agg_combine(W, G, P);
    }
    return pre_extend(X, G, P);                          // walked back to the very beginning
}

}  // namespace v7
}  // namespace dtk

#include "encode_v7_compact.cuh"
#include "encode_v7_scan.cuh"
#include "encode_v7_kernel.cuh"
