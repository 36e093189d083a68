// encode_v4.cuh -- single-pass classify + strip + {single-nt | k-mer} + CSR offsets over chained SUPER-TILES.
//
// One persistent CTA (256 threads, 4 per SM) claims flat super-tiles of S x 16 KiB input bytes in order (atomic
// ticket, fetched one super-tile ahead together with its record range and an L2 prefetch of its bytes).  The
// super-tile is the unit of the chained scan (decoupled look-back): the chain advances 32 super-tiles per L2 round
// trip, so its rate grows with S (profiles/r1_v3_encode.md: with 16 KiB units the chain, not HBM, was the bound).
// Inside the super-tile the CTA walks S sub-tiles; each thread owns 64 contiguous input bytes of the sub-tile,
// loaded straight into registers with four 16-byte loads.  Per sub-tile (two block barriers, no one-warp section):
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
// Per super-tile:
//   the entry line state comes from a chain of its own (one word per super-tile); the sub-tile loop runs under the
//      assumption IN_LINE and the (rare) super-tiles where that matters are redone;
//   P4 warp 0 publishes the aggregate, folds the 32 nearest predecessors in parallel (decoupled look-back) and
//      publishes the inclusive prefix; warp 6 builds the segment table, warp 7 prepares the next super-tile;
//   P5 tokens are cut from the stream in groups of 16 output bytes: one funnel-shift alignment per group,
//      windows at compile-time offsets, one 16-byte store straight to ids_out.
// Input bytes are read from HBM exactly once and ids written exactly once.
#pragma once
#include "common.cuh"

namespace dtk {

constexpr int NW = NT / 32;
constexpr int WB = 32 * LB;                  // input bytes per warp per sub-tile (2 KiB)
constexpr int PEND = 16;                     // stream slots in front of the super-tile's kept bases (carried bases)
constexpr int STREAM_BASES = PEND + S_MAX * TB;
constexpr int SW_CODE = (STREAM_BASES / 16 + 8 + 3) & ~3;
constexpr int SW_FLAG = (STREAM_BASES / 32 + 9 + 3) & ~3;
constexpr int SW_ALL = SW_CODE + SW_FLAG;    // multiple of 4 words
constexpr int EVW = 32;                      // record starts per super-tile handled by the one-warp path
constexpr int ENT_CAP = NT + 1;              // segment-table entries per emission pass

struct Smem4 {
    uint32_t strm[SW_ALL];                   // code stream: base u at word u>>4, bits 31-2(u&15), 30-2(u&15);
                                             // flag stream at strm + SW_CODE: base u at word u>>5, bit 31-(u&31)
    unsigned long long wk[NW][32];           // per warp: record-start bitmap of its 2 KiB (P1), then keep masks (P3)
    int32_t ent_src[ENT_CAP];                // segment table: stream position of the segment's first base
    int32_t ent_t[ENT_CAP];                  //   super-tile-relative index of its first token
    int32_t ent_nwin[ENT_CAP];               //   full windows available (tokens beyond are tail tokens)
    int32_t ev_p[2][EVW];                    // super-tile positions of the first EVW record starts (by parity)
    int32_t ev_k[EVW];                       // kept bases before each of them
    uint16_t offw[NW][32];                   // per warp: exclusive kept-base prefix of each lane
    int32_t warp_cnt[2][NW];                 // by sub-tile parity
    uint32_t warp_ls[2][NW];
    uint32_t ls_sub[2];                      // exit line state of the sub-tile (by sub-tile parity)
    int32_t scan_tmp[NW];
    uint8_t lut[256];
    // control of the current / next super-tile (by parity)
    int32_t c_tile[2], c_m[2];
    long long c_rlo[2];
    // per-super-tile scalars
    uint32_t t_ls, ls_in, redo;
    int32_t fk, lk, closed;                  // aggregate: kept before first / after last record start, tokens of records inside
    int32_t pend, tok0, ntok;                // carried bases, tokens of the open record's piece, tokens of the super-tile
    long long T0;                            // global index of the super-tile's first token
};
static_assert(sizeof(Smem4) <= 56 * 1024, "four CTAs per SM");

// ---------------------------------------------------------------------------------------- small helpers
__device__ __forceinline__ unsigned long long bit_at(int q) { return 0x8000000000000000ull >> q; }          // q in 0..63
__device__ __forceinline__ unsigned long long from_pos(int q) { return q >= 64 ? 0ull : (~0ull >> q); }   // positions >= q
__device__ __forceinline__ int first_pos(unsigned long long m) { return m ? __clzll((long long)m) : 64; }

__device__ __forceinline__ const uint32_t *flag_stream(const Smem4 &sm) { return sm.strm + SW_CODE; }

// k digits starting at base u (k <= 16)
__device__ __forceinline__ uint32_t code_at(const Smem4 &sm, int u, int k) {
    const int b = 2 * u, w = b >> 5, s = b & 31;
    return __funnelshift_l(sm.strm[w + 1], sm.strm[w], s) >> (32 - 2 * k);
}
__device__ __forceinline__ uint32_t flags_at(const Smem4 &sm, int u, int k) {    // k flag bits starting at base u
    const int w = u >> 5, s = u & 31;
    const uint32_t *f = flag_stream(sm);
    return __funnelshift_l(f[w + 1], f[w], s) >> (32 - k);
}
// class code 0..5 of base u: ACGT from the code plane; flagged bases carry digit 2 for N (what the arithmetic
// classification yields for 'N' / 'n') and digit 1 for UNK
__device__ __forceinline__ uint32_t class_at(const Smem4 &sm, int u) {
    const uint32_t c = code_at(sm, u, 1);
    return flags_at(sm, u, 1) ? (c == 2u ? CLS_N : CLS_UNK) : c;
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

// ---- emission ---------------------------------------------------------------------------------------
// One group = R = 16 / sizeof(IdT) consecutive output slots, aligned to 16 bytes in ids_out.  A thread that
// owns a full group inside the window part of one segment reads the stream words once, aligns them with one
// funnel shift per word and cuts R windows at compile-time offsets; everything else goes one token at a time.
template <typename IdT, int K, bool SINGLE>
__device__ __forceinline__ void emit_group_fast(const EncArgs &A, const Smem4 &sm, int u, IdT *dst, bool affine) {
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
        for (int i = 0; i <= NA; ++i) raw[i] = sm.strm[w + i];
#pragma unroll
        for (int i = 0; i < NA; ++i) a[i] = __funnelshift_l(raw[i + 1], raw[i], s);
    }
    uint32_t anybad = 0;
    {
        const int w = SW_CODE + (u >> 5), s = u & 31;
        uint32_t raw[NF + 1];
#pragma unroll
        for (int i = 0; i <= NF; ++i) raw[i] = sm.strm[w + i];
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
        else id[t] = P.base_id + (int32_t)c[t];
    }
    if (anybad) {
#pragma unroll
        for (int t = 0; t < R; ++t) {
            const int bo = K * t, i = bo >> 5, s = bo & 31;
            const uint32_t m = (s + K <= 32) ? ((f[i] >> (32 - s - K)) & ((1u << K) - 1u))
                                             : (__funnelshift_l(f[(i + 1 < NF) ? i + 1 : i], f[i], s) >> (32 - K));
            if (m) id[t] = (SINGLE && c[t] == 2u) ? P.nt_ids[4] : P.unk_id;
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
__device__ __forceinline__ void emit_token_slow(const EncArgs &A, const Smem4 &sm, int i, int j, int64_t gidx) {
    const EncParams &P = A.prm;
    const int jj = j - sm.ent_t[i], nwin = sm.ent_nwin[i], src = sm.ent_src[i];
    int32_t id;
    if (P.mode != MODE_KMER) {
        const uint32_t c = class_at(sm, src + jj);
        id = c <= CLS_N ? P.nt_ids[c] : P.unk_id;
    } else if (jj < nwin) {
        const int u = src + jj * P.k;
        id = flags_at(sm, u, P.k) ? P.unk_id : (int32_t)(P.base_id + code_at(sm, u, P.k));
    } else if (P.tail_policy == TAIL_PER_BASE) {
        const uint32_t c = class_at(sm, src + nwin * P.k + (jj - nwin));
        id = c <= CLS_N ? (int32_t)(P.base_id + P.four_k + c) : P.unk_id;
    } else {
        id = P.unk_id;
    }
    store_id<IdT>(A, gidx, id);
}

// largest i < nent with ent_t[i] <= j (ent_t is non-decreasing and ent_t[0] <= j)
__device__ __forceinline__ int find_ent(const Smem4 &sm, int nent, int j) {
    if (nent <= 4) {
        int i = 0;
        for (int e = 1; e < nent; ++e) i = (sm.ent_t[e] <= j) ? e : i;
        return i;
    }
    int lo = 0, hi = nent;
    while (hi - lo > 1) {
        const int mid = (lo + hi) >> 1;
        if (sm.ent_t[mid] <= j) lo = mid; else hi = mid;
    }
    return lo;
}

// tokens [ja, jb) (super-tile-relative) of the current segment table; `a` = T0 mod R, gbase = T0 - a
template <typename IdT>
__device__ __forceinline__ void emit_range(const EncArgs &A, const Smem4 &sm, int ja, int jb, int nent, int a,
                                           int64_t gbase, int cap_rel, bool vec_ok, bool affine) {
    constexpr int R = 16 / (int)sizeof(IdT);
    const EncParams &P = A.prm;
    const int kk = P.mode == MODE_KMER ? P.k : 0;        // 0: single-nt
    const int kstep = P.mode == MODE_KMER ? P.k : 1;
    IdT *idsA = reinterpret_cast<IdT *>(A.ids) + gbase;
    for (int q = (ja + a) / R + (int)threadIdx.x; q * R - a < jb; q += NT) {
        const int j0 = q * R - a;
        const int lo = j0 < ja ? ja : j0, hi = (j0 + R < jb) ? j0 + R : jb;
        int i = find_ent(sm, nent, lo);
        const int jj = lo - sm.ent_t[i];
        if (vec_ok && hi - lo == R && jj + R <= sm.ent_nwin[i] && q * R + R <= cap_rel) {
            const int u = sm.ent_src[i] + jj * kstep;
            IdT *dst = idsA + q * R;
            switch (kk) {
                case 0: emit_group_fast<IdT, 1, true>(A, sm, u, dst, affine); break;
                case 1: emit_group_fast<IdT, 1, false>(A, sm, u, dst, false); break;
                case 2: emit_group_fast<IdT, 2, false>(A, sm, u, dst, false); break;
                case 3: emit_group_fast<IdT, 3, false>(A, sm, u, dst, false); break;
                case 4: emit_group_fast<IdT, 4, false>(A, sm, u, dst, false); break;
                case 5: emit_group_fast<IdT, 5, false>(A, sm, u, dst, false); break;
                case 6: emit_group_fast<IdT, 6, false>(A, sm, u, dst, false); break;
                default: emit_group_fast<IdT, 8, false>(A, sm, u, dst, false); break;
            }
        } else {
            for (int j = lo; j < hi; ++j) {
                while (i + 1 < nent && sm.ent_t[i + 1] <= j) ++i;
                emit_token_slow<IdT>(A, sm, i, j, gbase + (int64_t)q * R + (j - j0));
            }
        }
    }
}

// ---- pre-pass: record range of every super-tile ----------------------------------------------------------
// first_rec[t] = first r in [0, n_rec] with position >= t * S * TB (n_rec + 1 if none); first_rec[n_tiles] = n_rec + 1
__global__ void __launch_bounds__(256) tile_first_rec_kernel(const __grid_constant__ EncArgs A) {
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

// ---- next-super-tile preparation (one warp): record range, record-start list, L2 prefetch of the bytes ----
__device__ __forceinline__ void prep_super(const EncArgs &A, Smem4 &sm, int par, unsigned long long ticket, int lane) {
    const unsigned long long rel = ticket - A.ticket_base;
    const int tile_n = rel >= (unsigned long long)A.n_tiles ? A.n_tiles : (int)rel;
    if (tile_n >= A.n_tiles) {
        if (lane == 0) sm.c_tile[par] = A.n_tiles;
        return;
    }
    const int64_t t0n = (int64_t)tile_n * A.S * TB;
    if (lane < A.S) {
        const int64_t b0 = t0n + (int64_t)lane * TB;
        int64_t sz = A.p_end - b0;
        sz = sz >= TB ? TB : ((sz + 15) & ~(int64_t)15);
        if (sz > 0)
            asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(A.bytes_al + b0), "r"((uint32_t)sz) : "memory");
    }
    const int64_t rlo = A.first_rec[tile_n], rhi = A.first_rec[tile_n + 1];
    const int64_t m64 = rhi - rlo;
    const int m = m64 > 0x7fffffff ? 0x7fffffff : (int)m64;
    if (m <= EVW && lane < m) sm.ev_p[par][lane] = (int)(rec_pos(A, rlo + lane) - t0n);
    if (lane == 0) { sm.c_tile[par] = tile_n; sm.c_m[par] = m; sm.c_rlo[par] = rlo; }
}

// exclusive block scan of one int per thread (two barriers)
__device__ __forceinline__ int block_exscan4(int v, Smem4 &sm, int &total) {
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

// ======================================================================================================
template <typename IdT>
__global__ void __launch_bounds__(NT, 4) encode_tiles_v4(const __grid_constant__ EncArgs A) {
    extern __shared__ __align__(16) uint8_t smem_raw[];
    Smem4 &sm = *reinterpret_cast<Smem4 *>(smem_raw);
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

    sm.lut[tid] = A.lut[tid];
    __syncthreads();
    unsigned long long next_ticket = 0;
    if (warp == NW - 1) {
        if (lane == 0) next_ticket = atomicAdd(A.ticket, 1ull);
        next_ticket = __shfl_sync(FULL, next_ticket, 0);
        prep_super(A, sm, 0, next_ticket, lane);
    }
    __syncthreads();

#pragma unroll 1
    for (int it = 0;; ++it) {
        const int par = it & 1;
        const int tile = sm.c_tile[par];
        if (tile >= A.n_tiles) break;
        const int m = sm.c_m[par];                             // record starts inside the super-tile
        const int64_t r_lo = sm.c_rlo[par];
        const int64_t t0 = (int64_t)tile * TBS;
        TileDesc &D = A.descs[tile];
        // sub-tiles that hold bytes or the position p_end (where the closing record offset may sit)
        const int64_t rem_b = A.p_end - t0;
        const int S_eff = rem_b >= TBS ? S : (int)(rem_b / TB) + 1;
        if (tid == (NW - 1) * 32) next_ticket = atomicAdd(A.ticket, 1ull);

        int ktot = 0;
        uint32_t ls_entry = LS_IN_LINE;
#pragma unroll 1
        for (int pass = 0;; ++pass) {
            // zero the stream (partial words are OR-ed in)
            {
                const int nb = PEND + S_eff * TB;
                const int c4 = ((nb >> 4) + 9 + 3) >> 2, f4 = ((nb >> 5) + 10 + 3) >> 2;
                uint4 *s4 = reinterpret_cast<uint4 *>(sm.strm);
                for (int i = tid; i < c4; i += NT) s4[i] = make_uint4(0, 0, 0, 0);
                for (int i = tid; i < f4; i += NT) s4[SW_CODE / 4 + i] = make_uint4(0, 0, 0, 0);
            }
            int base = 0;                                        // kept bases of the sub-tiles done so far
            uint32_t ls_use = ls_entry;                          // entry line state of the sub-tile
            uint32_t t_hr = 0, t_x = LS_LINE_START;              // line-state summary of the super-tile (warp NW-1)
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
#pragma unroll
                    for (int j = 0; j < 4; ++j)
                        v[j] = (full || p0 + 16 * j < A.p_end) ? __ldg(src + j) : make_uint4(0, 0, 0, 0);
                }
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
                        const int64_t lo_pos = t0 + wb, hi_pos = lo_pos + WB;
                        int lo = 0, hi = m;                          // first event at or after the warp's first byte
                        while (lo < hi) {
                            const int mid = (lo + hi) >> 1;
                            if (rec_pos(A, r_lo + mid) >= lo_pos) hi = mid; else lo = mid + 1;
                        }
                        e_lo = lo;
                        for (int e = e_lo; e < m; e += 32) {
                            const int ee = e + lane;
                            const int64_t pp = ee < m ? rec_pos(A, r_lo + ee) : hi_pos;
                            const uint32_t inr = __ballot_sync(FULL, pp < hi_pos);
                            if (inr && e_cnt == 0) { sm.wk[warp][lane] = 0ull; __syncwarp(); }
                            if (pp < hi_pos) atomicOr(&sm.wk[warp][(int)(pp - lo_pos) >> 6], bit_at((int)(pp - lo_pos) & 63));
                            e_cnt += __popc(inr);
                            if (inr != FULL) break;
                        }
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
                    E = flags_to_plane(fb);
                    if (!P.fast_lut) E = ~0ull;
                    bad = E;
                    // runs of N: classified arithmetically too (their digit is already 2), not one LUT trip per byte
                    if (P.fast_lut && P.fast_n && __any_sync(FULL, __popcll(E) >= 4)) {
#pragma unroll
                        for (int j = 0; j < 16; ++j) fb[j] = is_n_word(xw[j]);
                        E &= ~flags_to_plane(fb);
                    }
                }
                unsigned long long skip = 0, nl = 0, gt = 0;
                {
                    const uint8_t *vb = A.bytes_al + p0;
                    unsigned long long rem = E;
                    while (rem) {
                        const int q = __clzll((long long)rem);
                        const unsigned long long bq = bit_at(q);
                        rem ^= bq;
                        const uint32_t byte = (full || p0 + q < A.p_end) ? (uint32_t)__ldg(vb + q) : 0u;
                        const uint32_t c = sm.lut[byte];
                        if (byte == '\n') nl |= bq;
                        if (byte == '>') gt |= bq;
                        if (c == CLS_SKIP) skip |= bq;
                        if (c < CLS_N) bad &= ~bq;
                        const unsigned long long cc = c < CLS_N ? c : (c == CLS_N ? 2u : 1u);
                        const int sh = 62 - 2 * (q & 31);
                        if (q < 32) chi = (chi & ~(3ull << sh)) | (cc << sh);
                        else clo = (clo & ~(3ull << sh)) | (cc << sh);
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
                if (P.strip_headers) {
                    bool pend0;
                    const unsigned long long ls0 = settle(ls_base | bit_at(0), pend0);
                    if (pend0) s_x = LS_LINE_START;
                    else if (!ls0) s_x = LS_LINE_START;
                    else s_x = (gt & (ls0 & (~ls0 + 1ull))) ? LS_IN_HEADER : LS_IN_LINE;   // lowest set bit = last line start
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
#pragma unroll
                    for (int w = 0; w < NW - 1; ++w) {
                        const uint32_t v2 = sm.warp_ls[sp][w], g_hr = v2 >> 2, g_x = v2 & 3u;
                        if (w < warp) { z_x = ls_apply(g_hr, g_x, z_x); z_hr |= g_hr; }
                    }
                    uint32_t st_in = ls_apply(z_hr, z_x, ls_use);
                    if (tid == NT - 1) {                             // whole sub-tile: exit state, super-tile summary
                        z_x = ls_apply(s_hr, s_x, z_x); z_hr |= s_hr;
                        sm.ls_sub[sp] = ls_apply(z_hr, z_x, ls_use);
                        t_x = ls_apply(z_hr, z_x, t_x); t_hr |= z_hr;
                    }
                    st_in = ls_apply(e_hr, e_x, st_in);
                    bool pd;
                    const unsigned long long ls = settle(ls_base | (st_in == LS_LINE_START ? bit_at(0) : 0ull), pd);
                    unsigned long long hs = ls & gt;                 // header lines that start inside this thread's bytes
                    if (st_in == LS_IN_HEADER) {
                        const int a = first_pos(nl), b = first_pos(rs);
                        const int e = (b <= a) ? b - 1 : a;          // through the '\n', or up to a record start
                        if (e >= 0) hdr |= (e >= 63) ? ~0ull : ~from_pos(e + 1);
                    }
                    while (hs) {
                        const int h = __clzll((long long)hs);
                        hs &= ~bit_at(h);
                        const int a = first_pos(nl & from_pos(h)), b = first_pos(rs & from_pos(h + 1));
                        const int e = (b <= a) ? b - 1 : a;
                        hdr |= from_pos(h) & ((e >= 63) ? ~0ull : ~from_pos(e + 1));
                    }
                }
                unsigned long long keep = ~skip & ~hdr;
                if (p0 < pos_first || p0 + LB > pos_last) {
                    const int64_t a = pos_first - p0, b = pos_last - p0;        // in-record positions are [a, b)
                    const unsigned long long ma = a <= 0 ? ~0ull : from_pos((int)(a > 64 ? 64 : a));
                    const unsigned long long mb = b <= 0 ? 0ull : (b >= 64 ? ~0ull : ~from_pos((int)b));
                    keep &= ma & mb;
                }
                const int n = __popcll(keep);
                if (n == 0) { chi = clo = bad = 0ull; }
                else if (n != 64) {
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
#pragma unroll
                for (int d = 1; d < 32; d <<= 1) { const int t = __shfl_up_sync(FULL, inc, d); if (lane >= d) inc += t; }
                if (lane == 31) sm.warp_cnt[sp][warp] = inc;
                __syncthreads();                                     // ---- C: warp counts, sub-tile exit line state

                // ================= P3: stream append; kept-base index of the record starts =========================
                int woff = 0, ksub = 0;
#pragma unroll
                for (int w = 0; w < NW; ++w) { const int t = sm.warp_cnt[sp][w]; woff += (w < warp) ? t : 0; ksub += t; }
                if (n > 0) {
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
                            if (whole) sm.strm[cw0 + i] = cwv[i];
                            else if (cwv[i]) atomicOr(&sm.strm[cw0 + i], cwv[i]);
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
                            if (whole) sm.strm[fw0 + i] = bwv[i];
                            else if (bwv[i]) atomicOr(&sm.strm[fw0 + i], bwv[i]);
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
                        if (m <= EVW) sm.ev_k[e] = kidx; else A.rec_k[r_lo + e] = kidx;
                    }
                    __syncwarp();
                }
                base += ksub;
                if (P.strip_headers) ls_use = sm.ls_sub[sp];
            }
            ktot = base;
            if (P.strip_headers && tid == NT - 1) sm.t_ls = (t_hr << 2) | t_x;
            __syncthreads();                                         // ---- D: stream, record-start indices, summary

            // ---- warp 0: entry line state of the super-tile, on a chain of its own -----------------------------
            if (pass == 0 && warp == 0) {
                uint32_t redo = 0, state = LS_LINE_START;
                if (P.strip_headers) {
                    const uint32_t tagL = gen << 8;
                    const uint32_t tl = sm.t_ls, s_hr = tl >> 2, s_x = tl & 3u;
                    if (lane == 0) st_vol32(&A.ls[tile], tagL | ((s_hr ? LK_FINAL : LK_SUMMARY) << 2) | s_x);
                    bool ok = true;
                    if (tile > 0) {
                        uint32_t carry = LS_LINE_START; bool have_carry = false;
                        for (int bs = tile - 1;; bs -= 32) {
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
                                __nanosleep(64);
                            }
                            if (!ok) break;
                            // the value that survives is the farthest non-LINE_START one at or before the final tile
                            const uint32_t nb = __ballot_sync(FULL, val != LS_LINE_START && lane <= f);
                            if (nb) { carry = __shfl_sync(FULL, val, 31 - __clz(nb)); have_carry = true; }
                            if (f < 32) break;
                        }
                        state = have_carry ? carry : LS_LINE_START;
                    }
                    if (!ok && lane == 0) A.status[1] = 1u;
                    if (!s_hr && lane == 0) st_vol32(&A.ls[tile], tagL | (LK_FINAL << 2) | (state == LS_LINE_START ? s_x : state));
                    const bool reset_at_0 = m > 0 && (m <= EVW ? sm.ev_p[par][0] == 0 : rec_pos(A, r_lo) == t0);
                    redo = (state != LS_IN_LINE) && !reset_at_0;
                }
                if (lane == 0) { sm.ls_in = state; sm.redo = redo; }
            }
            // ---- warp NW-2: aggregate of the super-tile and the segment table of its record starts ---------------
            if (warp == NW - 2) {
                if (m == 0) {
                    if (lane == 0) { sm.fk = ktot; sm.lk = ktot; sm.closed = 0; sm.ntok = 0; }
                } else if (m <= EVW) {
                    const int ke = lane < m ? sm.ev_k[lane] : ktot;
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
                    const int tot = __shfl_sync(FULL, ti, 31), closed = __shfl_sync(FULL, ex, m - 1);
                    if (lane < m) { sm.ent_src[1 + lane] = PEND + ke; sm.ent_t[1 + lane] = ex; sm.ent_nwin[1 + lane] = nw; }
                    if (lane == 0) { sm.fk = ke; sm.closed = closed; sm.ntok = tot; }
                    if (lane == m - 1) sm.lk = ne;
                } else {
                    // many record starts: only the aggregate here, the table is built chunk by chunk in P5
                    int closed = 0, fk = 0;
                    for (int c0 = 0; c0 < m; c0 += 32) {
                        const int e = c0 + lane;
                        const int ke = e < m ? __ldcg(A.rec_k + r_lo + e) : ktot;
                        int kn = __shfl_down_sync(FULL, ke, 1);
                        if (lane == 31) kn = e + 1 < m ? __ldcg(A.rec_k + r_lo + e + 1) : ktot;
                        const int te = e < m - 1 ? tok_count32(kn - ke, P) : 0;
                        closed += __reduce_add_sync(FULL, te);
                        if (c0 == 0) fk = __shfl_sync(FULL, ke, 0);
                    }
                    if (lane == 0) {
                        sm.fk = fk; sm.closed = closed; sm.ntok = 0;
                        sm.lk = ktot - __ldcg(A.rec_k + r_lo + m - 1);
                    }
                }
            }
            __syncthreads();                                         // ---- D2: entry line state, aggregate
            if (pass == 1 || !sm.redo) break;
            ls_entry = sm.ls_in;
        }

        // ================= P4: warp 0 aggregate / look-back / inclusive prefix; warp 7 next super-tile =========
        if (warp == NW - 1) {
            next_ticket = __shfl_sync(FULL, next_ticket, 0);
            prep_super(A, sm, par ^ 1, next_ticket, lane);
        }
        if (warp == 0) {
            const uint32_t tagA = (gen << 2) | ST_AGG, tagI = (gen << 2) | ST_INCL;
            const int fk = sm.fk, lk = sm.lk, closed = sm.closed;
            const uint32_t hasev = m > 0;
            // last tn = min(k - 1, lk) classes of the super-tile, 3 bits each, newest lowest
            const int tn = min(k - 1, lk);
            unsigned long long gtail = 0;
            {
                unsigned long long tl = 0;
                if (lane < tn) tl = (unsigned long long)class_at(sm, PEND + ktot - tn + lane) << (3 * (tn - 1 - lane));
                gtail = ((unsigned long long)__reduce_or_sync(FULL, (uint32_t)(tl >> 32)) << 32) | __reduce_or_sync(FULL, (uint32_t)tl);
            }
            if (lane == 0) {
                st_vol128(&D.a0, make_uint4(tagA, (uint32_t)fk, (uint32_t)lk, (uint32_t)closed | (hasev << 31)));
                st_vol128(&D.a1, make_uint4(tagA, (uint32_t)tn | ((uint32_t)(gtail >> 32) << 4), (uint32_t)gtail, 0u));
            }
            // exclusive prefix of the super-tile
            int64_t XT = 0; QR Xo; Xo.q = 0; Xo.r = 0;
            unsigned long long xtail = 0;                        // last Xo.r classes of the open record
            if (tile > 0) {
                const int j = tile - 1 - lane;
                uint4 wa = make_uint4(0, 0, 0, 0), wb1 = wa, w0 = wa, w1 = wa;
                uint32_t st = ST_INCL;                           // tiles before 0 carry the empty inclusive prefix
                int f = 32; bool ok = true;
                for (int spins = 0;; ++spins) {
                    if (j >= 0) {
                        const TileDesc &Dj = A.descs[j];
                        w0 = ld_vol128(&Dj.i0); w1 = ld_vol128(&Dj.i1); wa = ld_vol128(&Dj.a0); wb1 = ld_vol128(&Dj.a1);
                        st = (w0.x == tagI && w1.x == tagI) ? ST_INCL : ((wa.x == tagA && wb1.x == tagA) ? ST_AGG : ST_EMPTY);
                    }
                    const uint32_t ib = __ballot_sync(FULL, st == ST_INCL);
                    f = ib ? __ffs(ib) - 1 : 32;                 // nearest tile with an inclusive prefix
                    const uint32_t missing = __ballot_sync(FULL, st == ST_EMPTY) & (f < 32 ? ((1u << f) - 1u) : FULL);
                    if (f < 32 && !missing) break;
                    if (spins > SPIN_LIMIT) { ok = false; break; }
                    __nanosleep(64);
                }
                if (!ok) { if (lane == 0) A.status[1] = 1u; f = 0; st = ST_INCL; w0 = w1 = make_uint4(0, 0, 0, 0); }
                // lanes < f hold aggregates (far = high lane), lane f the inclusive prefix they extend
                const bool in = lane < f;
                const int fk_l = in ? (int)wa.y : 0, lk_l = (int)wa.z, cl_l = (int)(wa.w & 0x7fffffffu);
                const bool ev_l = in && (wa.w >> 31);
                int Ps = fk_l;                                   // kept-before-first-start summed over lanes >= this one
#pragma unroll
                for (int d = 1; d < 32; d <<= 1) { const int t = __shfl_down_sync(FULL, Ps, d); if (lane + d < 32) Ps += t; }
                const uint32_t evmask = __ballot_sync(FULL, ev_l);
                const int64_t fT = (int64_t)(((uint64_t)w0.z << 32) | w0.y), fq = (int64_t)(((uint64_t)w1.z << 32) | w1.y);
                XT = __shfl_sync(FULL, fT, f);
                QR Fo; Fo.q = __shfl_sync(FULL, fq, f); Fo.r = (int32_t)(__shfl_sync(FULL, w0.w, f) & 15u);
                const int P0 = __shfl_sync(FULL, Ps, 0);
                if (!evmask) {
                    Xo = qr_add(Fo, qr_of((uint32_t)P0, P), k);
                } else {
                    const uint32_t higher = lane == 31 ? 0u : (evmask & ~((2u << lane) - 1u));
                    const int ep = higher ? __ffs(higher) - 1 : -1;          // next farther tile with a record start
                    const int P_ep = __shfl_sync(FULL, Ps, ep < 0 ? 0 : ep), lk_ep = __shfl_sync(FULL, lk_l, ep < 0 ? 0 : ep);
                    int t32 = 0; int64_t t64 = 0;
                    if (ev_l) {
                        if (ep >= 0) t32 = tok_count32(lk_ep + Ps - P_ep, P) + cl_l;
                        else t64 = qr_tokens(qr_add(Fo, qr_of((uint32_t)Ps, P), k), P) + cl_l;   // closes the record open at f
                    }
                    const int e1 = 31 - __clz(evmask), e0 = __ffs(evmask) - 1;
                    XT += __shfl_sync(FULL, t64, e1) + (int64_t)__reduce_add_sync(FULL, t32);
                    const int Pe0 = __shfl_sync(FULL, Ps, e0), lke0 = __shfl_sync(FULL, lk_l, e0);
                    Xo = qr_of((uint32_t)(lke0 + P0 - Pe0), P);
                }
                // pending classes of the open record: newest from the nearest tiles, older ones from farther back
                if (P.mode == MODE_KMER && Xo.r > 0) {
                    const unsigned long long mytail = st == ST_INCL ? ((unsigned long long)w1.w | ((unsigned long long)((w0.w >> 8) & 0x3ffu) << 32))
                                                                    : ((unsigned long long)wb1.z | ((unsigned long long)((wb1.y >> 4) & 0x3ffu) << 32));
                    const int mycnt = st == ST_INCL ? (int)((w0.w >> 4) & 15u) : (int)(wb1.y & 15u);
                    int have = 0;
                    for (int l = 0; l <= f && have < Xo.r; ++l) {
                        const unsigned long long tl = __shfl_sync(FULL, mytail, l);
                        const int cn = min(__shfl_sync(FULL, mycnt, l), Xo.r - have);
                        xtail |= (tl & ((1ull << (3 * cn)) - 1ull)) << (3 * have);
                        have += cn;
                        if (l < f && ((evmask >> l) & 1u)) break;
                    }
                }
            }
            // this super-tile's piece of the open record, inclusive prefix, segment-table entry 0
            const int pend = P.mode == MODE_KMER ? Xo.r : 0;
            const int nbase0 = pend + fk;
            const int nwin0 = (int)div_k((uint32_t)nbase0, P), rem0 = nbase0 - nwin0 * k;
            const int tok0 = nwin0 + (hasev ? tail_tokens(rem0, P) : 0);
            {
                int64_t YT; QR Yo; unsigned long long ytail; int ycnt;
                if (!hasev) {
                    YT = XT; Yo.q = Xo.q + nwin0; Yo.r = rem0;
                    const int keepx = min(Xo.r, k - 1 - tn);
                    ytail = ((xtail & ((1ull << (3 * keepx)) - 1ull)) << (3 * tn)) | gtail;
                    ycnt = keepx + tn;
                } else {
                    YT = XT + Xo.q + tok0 + closed; Yo = qr_of((uint32_t)lk, P); ytail = gtail; ycnt = tn;
                }
                if (lane == 0) {
                    st_vol128(&D.i0, make_uint4(tagI, (uint32_t)YT, (uint32_t)((uint64_t)YT >> 32),
                                                (uint32_t)Yo.r | ((uint32_t)ycnt << 4) | ((uint32_t)(ytail >> 32) << 8)));
                    st_vol128(&D.i1, make_uint4(tagI, (uint32_t)Yo.q, (uint32_t)((uint64_t)Yo.q >> 32), (uint32_t)ytail));
                }
            }
            // carried bases of the open record go in front of the stream
            {
                uint32_t cw = 0, fw = 0;
                if (lane < pend) {
                    const uint32_t c = (uint32_t)(xtail >> (3 * (pend - 1 - lane))) & 7u;
                    const int uu = PEND - pend + lane;
                    const uint32_t dg = c < CLS_N ? c : (c == CLS_N ? 2u : 1u);
                    cw = dg << (30 - 2 * uu);
                    fw = c >= CLS_N ? (1u << (31 - uu)) : 0u;
                }
                cw = __reduce_or_sync(FULL, cw); fw = __reduce_or_sync(FULL, fw);
                if (lane == 0) { sm.strm[0] = cw; if (fw) atomicOr(&sm.strm[SW_CODE], fw); }
            }
            if (m <= EVW && lane < m) sm.ent_t[1 + lane] += tok0;
            if (lane == 0) {
                sm.ent_src[0] = PEND - pend; sm.ent_t[0] = 0; sm.ent_nwin[0] = nwin0;
                sm.pend = pend; sm.tok0 = tok0; sm.ntok += tok0;
                sm.T0 = A.out_bias + XT + Xo.q;
            }
        }
        __syncthreads();                                         // ---- E: prefix known, next super-tile prepared

        // ================= P5: emit ============================================================================
        {
            const int64_t T0 = sm.T0;
            const int a = (int)(T0 & (R - 1));
            const int64_t gbase = T0 - a;
            const int64_t capl = A.ids_cap - gbase;
            const int cap_rel = capl < 0 ? 0 : (capl > 0x7fffffff ? 0x7fffffff : (int)capl);
            const int tok0 = sm.tok0;
            if (m <= EVW) {
                if (tid < m) A.out_off[r_lo + tid] = T0 + sm.ent_t[1 + tid];
                emit_range<IdT>(A, sm, 0, sm.ntok, m + 1, a, gbase, cap_rel, vec_ok, affine);
            } else {
                int tbase = tok0;                                // super-tile-relative token index of the chunk's first record
                for (int c0 = 0; c0 < m; c0 += NT) {
                    const int cm = min(NT, m - c0), e = c0 + tid;
                    int ke = ktot, ne = 0, te = 0, nw = 0;
                    if (e < m) {
                        ke = __ldcg(A.rec_k + r_lo + e);
                        const int kn = e + 1 < m ? __ldcg(A.rec_k + r_lo + e + 1) : ktot;
                        ne = kn - ke;
                        nw = (int)div_k((uint32_t)ne, P);
                        te = e + 1 < m ? nw + tail_tokens(ne - nw * k, P) : nw;
                    }
                    int total;
                    const int ex = block_exscan4(te, sm, total);
                    if (e < m) {
                        sm.ent_src[1 + tid] = PEND + ke; sm.ent_t[1 + tid] = tbase + ex; sm.ent_nwin[1 + tid] = nw;
                        A.out_off[r_lo + e] = T0 + tbase + ex;
                    }
                    if (c0 > 0 && tid == 0) { sm.ent_src[0] = 0; sm.ent_t[0] = tbase; sm.ent_nwin[0] = 0; }
                    __syncthreads();
                    emit_range<IdT>(A, sm, c0 == 0 ? 0 : tbase, tbase + total, cm + 1, a, gbase, cap_rel, vec_ok, affine);
                    tbase += total;
                    __syncthreads();
                }
            }
        }
        __syncthreads();                                         // ---- A: stream and tables free for the next super-tile
    }
}

}  // namespace dtk
