// encode_v8.cuh -- single-pass classify + strip + {single-nt | k-mer} + CSR offsets with a BARRIER-FREE byte loop.
//
// Same outer structure as encode_v5.cuh (persistent CTAs, super-tiles of S x 16 KiB claimed by ticket, the chained scan
// with decoupled look-back, loop(B) -> aggregate(B) -> look-back(A) -> emit(A)), and the same classification, line-state
// algebra and emission arithmetic; what changes is everything between the loads and the emission:
//   * every WARP owns whole 2 KiB chunks of the super-tile (chunk c = s * 8 + warp) and never waits for another warp
//     inside the loop: the kept bases of a chunk are compacted inside the warp (shuffle scan) and stored in the chunk's
//     own SLOT of the kept-base stream (128 code words + 64 flag words, left-aligned); the per-chunk counts are scanned
//     once per super-tile by one warp.  Emission maps a stream position to (slot, offset) through that prefix array.
//     A 16-byte output group that lies inside one slot is cut exactly as in v5; the few groups that straddle two slots
//     are assembled token by token.
//   * the entry line state of a chunk is read off the 128 bytes in front of it (a newline or a record start inside that
//     window settles it: always the case for wrapped FASTA).  If the window does not settle it the chunk assumes IN_LINE
//     and raises a flag; such super-tiles compose their chunk summaries after the loop (one warp), compare every chunk's
//     true entry state with the one it used and redo the loop with the true states when they differ.
//   * slot words are written exactly once (the bits a lane shares with its neighbour travel by shuffle), so the stream
//     needs no zeroing and no shared-memory atomics on the common path.
// One block barrier per super-tile pass instead of two per 16 KiB.
#pragma once
#include "encode_v5.cuh"

namespace dtk {
namespace v8 {

using namespace dtk::v5;

constexpr int NCH = S_MAX * NW;                  // chunks (slots) per super-tile, at most
constexpr int CWS = WB / 16;                     // code words per slot (2 bits per base)
constexpr int FWS = WB / 32;                     // flag words per slot
constexpr int S0W = 4;                           // words of slot 0 (the carried bases: word 0 only)
constexpr int SW8_CODE = S0W + NCH * CWS + 4;    // + over-read slack
constexpr int SW8_FLAG = S0W + NCH * FWS + 4;
constexpr int SW8_ALL = SW8_CODE + SW8_FLAG;
static_assert(SW8_ALL % 4 == 0, "stream buffers stay 16-byte aligned");
static_assert(WB == 2048, "locate() shifts by 11");

struct Smem8 {
    uint32_t strm[2][SW8_ALL];                   // per buffer: code words of slot 0, slots 1..NCH, then the flag words
    unsigned long long wk[NW][32];               // per warp: record-start bitmap of its chunk, then keep masks
    int32_t ent_src[ENT_CAP];                    // many-starts segment table (see encode_v5.cuh)
    int32_t ent_t[ENT_CAP];
    int32_t ent_nwin[ENT_CAP];
    int32_t seg_src[2][EVW + 1];
    int32_t seg_t[2][EVW + 1];
    int32_t seg_nwin[2][EVW + 1];
    int32_t ev_p[2][EVW];                        // super-tile positions of the first EVW record starts (by ticket parity)
    int32_t ev_k[2][EVW];                        // kept bases before each of them (chunk-relative until the aggregate warp ran)
    uint16_t offw[NW][32];
    int32_t pre[2][NCH + 2];                     // per buffer: stream position of slot t's first base; [NCH + 1] = end
    int32_t cnt[NCH];                            // kept bases of every chunk of super-tile B
    uint8_t sum[NCH];                            // line-state summary of every chunk: has_reset << 2 | exit state
    uint8_t ent_used[NCH];                       // entry line state the chunk ran with
    uint8_t ent_true[NCH];                       // entry line states for the redo pass
    int32_t scan_tmp[NW];
    uint8_t lut[256];
    TileAgg ag[2];
    int32_t c_tile[2], c_m[2];
    uint32_t c_ls[2];
    long long c_rlo[2];
    uint32_t assumed[2];                         // by ticket parity: some chunk assumed its entry line state
    uint32_t redo;
    int32_t tok0, ntok;
    long long T0;
};
static_assert(sizeof(Smem8) <= 56 * 1024, "shared memory per CTA (4 CTAs per SM)");

// ---- stream access through the slot prefix ---------------------------------------------------------------
struct Strm { const uint32_t *st; const int32_t *pre; };

__device__ __forceinline__ int cbase(int t) { return t ? S0W + (t - 1) * CWS : 0; }
__device__ __forceinline__ int fbase(int t) { return SW8_CODE + (t ? S0W + (t - 1) * FWS : 0); }

// slot t and offset o of stream position u (0 <= u < end of the stream)
__device__ __forceinline__ int locate(const int32_t *pre, int u, int &o) {
    int t = u < PEND ? 0 : 1 + ((u - PEND) >> 11);
    while (t < NCH && u >= pre[t + 1]) ++t;
    o = u - pre[t];
    return t;
}

// nb <= 15 bases starting at stream position u: 2 nb code bits and nb flag bits (slot by slot)
__device__ __forceinline__ void gather_bases(const Strm &Z, int u, int nb, uint32_t &code, uint32_t &flag) {
    int o;
    int t = locate(Z.pre, u, o);
    code = 0u; flag = 0u;
    int got = 0;
    for (;;) {
        const int take = min(Z.pre[t + 1] - Z.pre[t] - o, nb - got);
        if (take > 0) {
            const uint32_t *cw = Z.st + cbase(t), *fw = Z.st + fbase(t);
            const int b = 2 * o;
            const uint32_t c = __funnelshift_l(cw[(b >> 5) + 1], cw[b >> 5], b & 31) >> (32 - 2 * take);
            const uint32_t f = __funnelshift_l(fw[(o >> 5) + 1], fw[o >> 5], o & 31) >> (32 - take);
            code = (code << (2 * take)) | c; flag = (flag << take) | f;
            got += take;
        }
        if (got >= nb || t >= NCH) break;
        ++t; o = 0;
    }
}
__device__ __forceinline__ uint32_t class_at8(const Strm &Z, int u) {
    uint32_t c, f;
    gather_bases(Z, u, 1, c, f);
    return f ? (c == 2u ? CLS_N : CLS_UNK) : c;
}

// ---- emission ---------------------------------------------------------------------------------------------
// One group of R = 16 / sizeof(IdT) output slots whose bases all lie in one slot (code words cw, flag words fw,
// first base at offset o): see emit_group_fast of encode_v5.cuh.
template <typename IdT, int K, bool SINGLE>
__device__ __forceinline__ void emit_group8(const EncArgs &A, const uint32_t *cw, const uint32_t *fw, int o, IdT *dst, bool affine) {
    constexpr int R = 16 / (int)sizeof(IdT);
    constexpr int W = 2 * K;
    constexpr int CB = W * R;
    constexpr int NA = (CB + 31) / 32;
    constexpr int FB = K * R;
    constexpr int NF = (FB + 31) / 32;
    const EncParams &P = A.prm;
    uint32_t a[NA], f[NF];
    {
        const int b = 2 * o, w = b >> 5, s = b & 31;
        uint32_t raw[NA + 1];
#pragma unroll
        for (int i = 0; i <= NA; ++i) raw[i] = cw[w + i];
#pragma unroll
        for (int i = 0; i < NA; ++i) a[i] = __funnelshift_l(raw[i + 1], raw[i], s);
    }
    uint32_t anybad = 0;
    {
        const int w = o >> 5, s = o & 31;
        uint32_t raw[NF + 1];
#pragma unroll
        for (int i = 0; i <= NF; ++i) raw[i] = fw[w + i];
#pragma unroll
        for (int i = 0; i < NF; ++i) {
            f[i] = __funnelshift_l(raw[i + 1], raw[i], s);
            const int lo = i * 32;
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

// one token made of the kk bases at stream position u (kk = 1: a single-nt token), gathered slot by slot
template <typename IdT, bool SINGLE>
__device__ __forceinline__ int32_t window_id8(const EncArgs &A, const Strm &Z, int u, int kk) {
    const EncParams &P = A.prm;
    uint32_t c, f;
    gather_bases(Z, u, kk, c, f);
    if (SINGLE) return f ? (c == 2u ? P.nt_ids[4] : P.unk_id) : P.nt_ids[c];
    return f ? P.unk_id : (int32_t)(P.base_id + c);
}

// token j (super-tile-relative) of segment-table entry i, any k
template <typename IdT>
__device__ __forceinline__ void emit_token_slow8(const EncArgs &A, const Strm &Z, const SegTab &G, int i, int j, int64_t gidx) {
    const EncParams &P = A.prm;
    const int jj = j - G.t[i], nwin = G.nwin[i], src = G.src[i];
    int32_t id;
    if (P.mode != MODE_KMER) {
        const uint32_t c = class_at8(Z, src + jj);
        id = c <= CLS_N ? P.nt_ids[c] : P.unk_id;
    } else if (jj < nwin) {
        id = window_id8<IdT, false>(A, Z, src + jj * P.k, P.k);
    } else if (P.tail_policy == TAIL_PER_BASE) {
        const uint32_t c = class_at8(Z, src + nwin * P.k + (jj - nwin));
        id = c <= CLS_N ? (int32_t)(P.base_id + P.four_k + c) : P.unk_id;
    } else {
        id = P.unk_id;
    }
    store_id<IdT>(A, gidx, id);
}

// one full group of R window tokens starting at stream position u, written with one 16-byte store
template <typename IdT, int K, bool SINGLE>
__device__ __forceinline__ void emit_group_at(const EncArgs &A, const Strm &Z, int u, IdT *dst, bool affine) {
    constexpr int R = 16 / (int)sizeof(IdT);
    constexpr int KS = SINGLE ? 1 : K;
    int o;
    const int t = locate(Z.pre, u, o);
    if (o + KS * R <= Z.pre[t + 1] - Z.pre[t]) {
        emit_group8<IdT, K, SINGLE>(A, Z.st + cbase(t), Z.st + fbase(t), o, dst, affine);
    } else {
        // the group straddles two slots (or sits on the carried bases): token by token, still one aligned store
        uint32_t p[4] = {0u, 0u, 0u, 0u};
#pragma unroll 1
        for (int x = 0; x < R; ++x) {
            const uint32_t id = (uint32_t)window_id8<IdT, SINGLE>(A, Z, u + x * KS, KS);
            const int per = 4 / (int)sizeof(IdT);                       // ids per 32-bit word
            const uint32_t v = sizeof(IdT) == 4 ? id : (sizeof(IdT) == 2 ? (id & 0xffffu) : (id & 0xffu));
            p[x / per] |= v << (8 * (int)sizeof(IdT) * (x % per));
        }
        *reinterpret_cast<uint4 *>(dst) = make_uint4(p[0], p[1], p[2], p[3]);
    }
}

template <typename IdT, int KK>
__device__ __forceinline__ void emit_group_switch(const EncArgs &A, const Strm &Z, int u, IdT *dst, bool affine, int kk) {
    if constexpr (KK == 0) emit_group_at<IdT, 1, true>(A, Z, u, dst, affine);
    else if constexpr (KK > 0) emit_group_at<IdT, KK, false>(A, Z, u, dst, false);
    else switch (kk) {
        case 0: emit_group_at<IdT, 1, true>(A, Z, u, dst, affine); break;
        case 1: emit_group_at<IdT, 1, false>(A, Z, u, dst, false); break;
        case 2: emit_group_at<IdT, 2, false>(A, Z, u, dst, false); break;
        case 3: emit_group_at<IdT, 3, false>(A, Z, u, dst, false); break;
        case 4: emit_group_at<IdT, 4, false>(A, Z, u, dst, false); break;
        case 5: emit_group_at<IdT, 5, false>(A, Z, u, dst, false); break;
        case 6: emit_group_at<IdT, 6, false>(A, Z, u, dst, false); break;
        default: emit_group_at<IdT, 8, false>(A, Z, u, dst, false); break;
    }
}

// tokens [ja, jb) (super-tile-relative) of the segment table G; `a` = T0 mod R, gbase = T0 - a   (many-starts path)
template <typename IdT, int KK>
__device__ __forceinline__ void emit_range8(const EncArgs &A, const Strm &Z, const SegTab &G, int ja, int jb, int nent, int a,
                                            int64_t gbase, int cap_rel, bool vec_ok, bool affine) {
    constexpr int R = 16 / (int)sizeof(IdT);
    const EncParams &P = A.prm;
    const int kk = P.mode == MODE_KMER ? P.k : 0;
    const int kstep = P.mode == MODE_KMER ? P.k : 1;
    IdT *idsA = reinterpret_cast<IdT *>(A.ids) + gbase;
    for (int q = (ja + a) / R + (int)threadIdx.x; q * R - a < jb; q += NT) {
        const int j0 = q * R - a;
        const int lo = j0 < ja ? ja : j0, hi = (j0 + R < jb) ? j0 + R : jb;
        int i = find_ent(G, nent, lo);
        const int jj = lo - G.t[i];
        if (vec_ok && hi - lo == R && jj + R <= G.nwin[i] && q * R + R <= cap_rel) {
            emit_group_switch<IdT, KK>(A, Z, G.src[i] + jj * kstep, idsA + q * R, affine, kk);
        } else {
            for (int j = lo; j < hi; ++j) {
                while (i + 1 < nent && G.t[i + 1] <= j) ++i;
                emit_token_slow8<IdT>(A, Z, G, i, j, gbase + (int64_t)q * R + (j - j0));
            }
        }
    }
}

// all tokens [0, ntok) of a short segment table (at most EVW + 1 entries)
template <typename IdT, int KK>
__device__ __forceinline__ void emit_segments8(const EncArgs &A, const Strm &Z, const SegTab &G, int nent, int ntok, int a,
                                               int64_t gbase, int cap_rel, bool vec_ok, bool affine) {
    constexpr int R = 16 / (int)sizeof(IdT);
    const EncParams &P = A.prm;
    const int kk = P.mode == MODE_KMER ? P.k : 0;
    const int ks = P.mode == MODE_KMER ? P.k : 1;
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
            for (int q = qa + (int)threadIdx.x; q < qb; q += NT)
                emit_group_switch<IdT, KK>(A, Z, u0 + (q * R - a - t_lo) * ks, idsA + q * R, affine, kk);
            const int h1 = min(t_hi, qa * R - a), h2 = max(t_lo, qb * R - a);     // tokens before / after the fast groups
            const int n1 = h1 - t_lo, n2 = t_hi - h2;
            for (int x = (int)threadIdx.x; x < n1 + n2; x += NT) {
                const int j = x < n1 ? t_lo + x : h2 + (x - n1);
                emit_token_slow8<IdT>(A, Z, G, i, j, gbase + a + j);
            }
        } else {
            for (int j = t_lo + (int)threadIdx.x; j < t_hi; j += NT) emit_token_slow8<IdT>(A, Z, G, i, j, gbase + a + j);
        }
    }
}

// ---- entry line state of the chunk that starts at super-tile offset cbo (global position pos), read off the 128 bytes
// in front of it (wv: lane l holds bytes 4l .. 4l+3 of that window).  LS_UNKNOWN when the window holds neither a newline
// nor the start of the record.  Same rule as prep_super of encode_v5.cuh.
__device__ __forceinline__ uint32_t window_entry(const EncArgs &A, const uint8_t *lut, uint32_t wv, int64_t pos, int cbo,
                                                 const int32_t *evp, int m, int64_t r_lo, int64_t t0, int lane,
                                                 int64_t pos_first, int64_t pos_last) {
    constexpr uint32_t FULL = 0xffffffffu;
    if (pos <= pos_first || pos >= pos_last) return LS_LINE_START;        // no record byte on one side: irrelevant
    int rsw = -1;                                                         // window index of the record's first byte
    if (m > 0) {
        int pl = -1;                                                      // last record start at or before the chunk
        if (m <= EVW) {
            const int p = lane < m ? evp[lane] : 0x7fffffff;
            const uint32_t bal = __ballot_sync(FULL, p <= cbo);
            if (bal) pl = __shfl_sync(FULL, p, 31 - __clz(bal));
        } else {
            int lo = 0, hi = m;                                           // number of record starts <= cbo
            while (lo < hi) {
                const int mid = (lo + hi) >> 1;
                if (rec_pos(A, r_lo + mid) - t0 <= cbo) lo = mid + 1; else hi = mid;
            }
            if (lo > 0) pl = (int)(rec_pos(A, r_lo + lo - 1) - t0);
        }
        if (pl == cbo) return LS_LINE_START;                              // a record starts right here
        if (pl >= 0) rsw = pl - (cbo - 128);
    }
    // newline, '>' and "not skippable" bits of this lane's four bytes; bytes the arithmetic proves to be ACGT are
    // none of the first two and never skippable
    uint32_t nlm = 0, gtm = 0, nsk = 0xfu;
    {
        uint32_t code, fl;
        classify_word(wv, code, fl);
        if (!A.prm.fast_lut) fl = 0x80808080u;
        while (fl) {
            const int i = (__ffs(fl) - 1) >> 3;
            fl &= fl - 1;
            const uint32_t byte = (wv >> (8 * i)) & 255u;
            nlm |= (uint32_t)(byte == '\n') << i;
            gtm |= (uint32_t)(byte == '>') << i;
            if (lut[byte] == CLS_SKIP && byte != '>') nsk &= ~(1u << i);   // '>' opens a header even if the table skips it
        }
    }
    int pstar = -1;                                                       // window index of the last line start
    const uint32_t nlb = __ballot_sync(FULL, nlm != 0);
    if (nlb) {
        const int L = 31 - __clz(nlb);
        const uint32_t mm = __shfl_sync(FULL, nlm, L);
        pstar = 4 * L + (31 - __clz(mm)) + 1;
    }
    if (rsw >= 0 && rsw > pstar) pstar = rsw;
    if (pstar < 0) return LS_UNKNOWN;
    uint32_t msk = nsk;
    const int lo = pstar - 4 * lane;                                      // this lane's bytes i >= lo count
    if (lo > 0) msk &= lo >= 4 ? 0u : (0xfu << lo);
    const uint32_t nb = __ballot_sync(FULL, msk != 0);
    if (!nb) return LS_LINE_START;
    const int L = __ffs(nb) - 1;
    const uint32_t mm = __shfl_sync(FULL, msk, L), gg = __shfl_sync(FULL, gtm, L);
    return ((gg >> (__ffs(mm) - 1)) & 1u) ? LS_IN_HEADER : LS_IN_LINE;
}

// inclusive warp scan of line-state summaries (hr, x): lane l ends up with the composition of lanes 0..l
__device__ __forceinline__ void ls_scan(uint32_t &hr, uint32_t &x, int lane) {
    constexpr uint32_t FULL = 0xffffffffu;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const uint32_t o_hr = __shfl_up_sync(FULL, hr, d), o_x = __shfl_up_sync(FULL, x, d);
        if (lane >= d) { x = ls_apply(hr, x, o_x); hr |= o_hr; }
    }
}

// ======================================================================================================
// KK: the emission variant compiled in -- 0 single-nt, 1..6 / 8 that k, -1 every variant behind a run-time switch
template <typename IdT, int KK>
__global__ void __launch_bounds__(NT, 1024 / NT) encode_tiles_v8(const __grid_constant__ EncArgs A) {
    extern __shared__ __align__(16) uint8_t smem_raw[];
    Smem8 &sm = *reinterpret_cast<Smem8 *>(smem_raw);
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
    if (tid < 2) sm.assumed[tid] = 0u;
    __syncthreads();
    unsigned long long next_ticket = 0;
    if (warp == NW - 1) {
        if (lane == 0) next_ticket = atomicAdd(A.ticket, 1ull);
        next_ticket = __shfl_sync(FULL, next_ticket, 0);
        prep_super(A, sm, 0, next_ticket, lane, pos_first, pos_last);
    }
    __syncthreads();

    bool haveA = false;
    int tileA = 0, mA = 0;
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
        int nch = 0;

        if (haveB) {
            const int64_t rem_b = A.p_end - t0;
            const int S_eff = rem_b >= TBS ? S : (int)(rem_b / TB) + 1;
            nch = S_eff * NW;
            const uint32_t ls_known = sm.c_ls[par];
            if (tid == (NW - 1) * 32) next_ticket = atomicAdd(A.ticket, 1ull);
            if (P.strip_headers && tid == 0 && ls_known == LS_UNKNOWN) sm.assumed[par] = 1u;
#pragma unroll 1
            for (int pass = 0;; ++pass) {
#pragma unroll 1
                for (int s = 0; s < S_eff; ++s) {
                    const int c = s * NW + warp;                          // this warp's chunk
                    const int cbo = c * WB;                               // super-tile offset of its first byte
                    const int64_t ts0 = t0 + (int64_t)s * TB;
                    const int64_t p0 = t0 + cbo + lane * LB;              // position of this thread's first byte
                    const bool full = ts0 + TB <= A.p_end;
                    // ================= load, classify, exceptions ==============================================
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
                    uint32_t wv = 0u;                                     // the 128 bytes in front of the chunk
                    const bool use_win = P.strip_headers && pass == 0 && c > 0;
                    if (use_win) {
                        const int64_t wp = t0 + cbo - 128 + 4 * lane;
                        if (wp < A.p_end) wv = __ldg(reinterpret_cast<const uint32_t *>(A.bytes_al + wp));
                    }
                    if (tid == 0 && s + 2 < S_eff) prefetch_l2(A, ts0 + 2 * TB);
                    // record starts inside this chunk: events [e_lo, e_lo + e_cnt) of the super-tile
                    int e_lo = 0, e_cnt = 0;
                    unsigned long long rs = 0ull;
                    if (m > 0) {
                        if (m <= EVW) {
                            const int p = lane < m ? sm.ev_p[par][lane] - cbo : -1;
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
                            e_cnt = warp_events_many(A, sm.wk[warp], r_lo, m, t0 + cbo, lane, e_lo);
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
                            if (byte == '\n') nl |= bq;
                            if (byte == '>') gt |= bq;
                            if (sm.lut[byte] == CLS_SKIP) skip |= bq;
                        }
                    }
                    // ================= line state: entry state of the chunk, header mask, chunk summary ===============
                    unsigned long long hdr = 0;
                    if (P.strip_headers) {
                        const unsigned long long osk = skip & ~nl & ~gt;   // SKIP bytes that neither end nor start a line
                        const uint32_t b_hard = __ballot_sync(FULL, (gt | osk) != 0ull);
                        const uint32_t b_reset = __ballot_sync(FULL, (nl | rs) != 0ull);
                        uint32_t ent;
                        if (pass) ent = sm.ent_true[c];
                        else if (c == 0) ent = ls_known == LS_UNKNOWN ? LS_IN_LINE : ls_known;
                        else {
                            ent = window_entry(A, sm.lut, wv, t0 + cbo, cbo, sm.ev_p[par], m, r_lo, t0, lane, pos_first, pos_last);
                            if (ent == LS_UNKNOWN) { ent = LS_IN_LINE; if (lane == 0) sm.assumed[par] = 1u; }
                        }
                        uint32_t c_hr, c_x;                                // summary of the whole chunk
                        if (!b_hard) {
                            // no '>' and no other SKIP byte in the chunk: no header starts here, and after the last line
                            // reset the line is open unless the chunk's last byte is that newline
                            c_hr = b_reset != 0u;
                            c_x = __shfl_sync(FULL, (uint32_t)(nl & 1ull), 31) ? LS_LINE_START : LS_IN_LINE;
                            if (ent == LS_IN_HEADER) {                     // the header runs to the chunk's first reset
                                if (!b_reset) hdr = ~0ull;
                                else {
                                    const int L = __ffs(b_reset) - 1;
                                    if (lane < L) hdr = ~0ull;
                                    else if (lane == L) {
                                        const int a = first_pos(nl), bb = first_pos(rs);
                                        const int e = (bb <= a) ? bb - 1 : a;     // through the '\n', or up to a record start
                                        if (e >= 0) hdr = (e >= 63) ? ~0ull : ~from_pos(e + 1);
                                    }
                                }
                            }
                        } else {
                            const unsigned long long ls_base = (nl >> 1) | rs;     // line starts: after each '\n', at record starts
                            auto settle = [&](unsigned long long ls, bool &pending) {
                                pending = (nl & 1ull) != 0;
                                unsigned long long t;
                                while ((t = ls & osk) != 0) { pending = pending || (t & 1ull); ls = (ls & ~t) | (t >> 1); }
                                return ls;
                            };
                            uint32_t s_hr = (nl | rs) != 0ull, s_x;
                            if ((gt | osk) == 0ull) s_x = (nl & 1ull) ? LS_LINE_START : LS_IN_LINE;
                            else {
                                bool pend0;
                                const unsigned long long ls0 = settle(ls_base | bit_at(0), pend0);
                                if (pend0 || !ls0) s_x = LS_LINE_START;
                                else s_x = (gt & (ls0 & (~ls0 + 1ull))) ? LS_IN_HEADER : LS_IN_LINE;
                            }
                            ls_scan(s_hr, s_x, lane);
                            c_hr = __shfl_sync(FULL, s_hr, 31); c_x = __shfl_sync(FULL, s_x, 31);
                            uint32_t e_hr = __shfl_up_sync(FULL, s_hr, 1), e_x = __shfl_up_sync(FULL, s_x, 1);
                            if (lane == 0) { e_hr = 0; e_x = LS_LINE_START; }
                            const uint32_t st_in = ls_apply(e_hr, e_x, ent);
                            if ((nl | gt | rs) == 0ull) {                  // no line ends or starts here: all header or none
                                if (st_in == LS_IN_HEADER) hdr = ~0ull;
                            } else if (gt == 0ull && st_in != LS_IN_HEADER) {
                                // no '>' here and not inside a header: nothing of this thread's bytes is header
                            } else {
                                bool pd;
                                const unsigned long long ls = settle(ls_base | (st_in == LS_LINE_START ? bit_at(0) : 0ull), pd);
                                unsigned long long hs = ls & gt;           // header lines that start inside this thread's bytes
                                if (st_in == LS_IN_HEADER) {
                                    const int a = first_pos(nl), bb = first_pos(rs);
                                    const int e = (bb <= a) ? bb - 1 : a;
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
                        if (lane == 0) { sm.sum[c] = (uint8_t)((c_hr << 2) | c_x); sm.ent_used[c] = (uint8_t)ent; }
                    }
                    // ================= keep mask, class of the kept exceptions, compaction =============================
                    unsigned long long keep = ~skip & ~hdr;
                    if (p0 < pos_first || p0 + LB > pos_last) {
                        const int64_t a = pos_first - p0, bb = pos_last - p0;       // in-record positions are [a, bb)
                        const unsigned long long ma = a <= 0 ? ~0ull : from_pos((int)(a > 64 ? 64 : a));
                        const unsigned long long mb = bb <= 0 ? 0ull : (bb >= 64 ? ~0ull : ~from_pos((int)bb));
                        keep &= ma & mb;
                    }
                    {
                        const uint8_t *vb = A.bytes_al + p0;
                        unsigned long long rem = E & keep;
                        while (rem) {
                            const int q = __clzll((long long)rem);
                            const unsigned long long bq = bit_at(q);
                            rem ^= bq;
                            const uint32_t byte = (full || p0 + q < A.p_end) ? (uint32_t)__ldg(vb + q) : 0u;
                            const uint32_t cl = sm.lut[byte];
                            if (cl < CLS_N) bad &= ~bq;
                            const unsigned long long cc = cl < CLS_N ? cl : (cl == CLS_N ? 2u : 1u);
                            const int sh = 62 - 2 * (q & 31);
                            if (q < 32) chi = (chi & ~(3ull << sh)) | (cc << sh);
                            else clo = (clo & ~(3ull << sh)) | (cc << sh);
                        }
                    }
                    const bool wfull = __all_sync(FULL, keep == ~0ull);  // nothing dropped in this chunk
                    const int n = __popcll(keep);
                    if (n == 0) { chi = clo = bad = 0ull; }
                    else if (n == 63) {
                        const int lo = __ffsll((long long)~keep) - 1;                      // plane bit of the dropped byte
                        const unsigned long long lm = (1ull << lo) - 1ull;
                        bad = (bad & ~(lm | (1ull << lo))) | ((bad & lm) << 1);
                        if (lo >= 32) {
                            const int pb = 2 * lo - 64;
                            const unsigned long long up = pb + 2 < 64 ? (~0ull << (pb + 2)) : 0ull;
                            chi = (chi & up) | ((chi & ((1ull << pb) - 1ull)) << 2) | (clo >> 62);
                            clo <<= 2;
                        } else {
                            const int pb = 2 * lo;
                            const unsigned long long up = pb + 2 < 64 ? (~0ull << (pb + 2)) : 0ull;
                            clo = (clo & up) | ((clo & ((1ull << pb) - 1ull)) << 2);
                        }
                    } else if (n != 64) {
                        unsigned long long drop = ~keep;
                        while (drop) {
                            const int lo = __ffsll((long long)drop) - 1;
                            const unsigned long long t = ~(drop >> lo);
                            const int len = t ? __ffsll((long long)t) - 1 : 64 - lo;
                            const unsigned long long lm = (1ull << lo) - 1ull;
                            const unsigned long long hm = (lo + len >= 64) ? 0ull : (~0ull << (lo + len));
                            drop &= hm;
                            bad = (bad & hm) | ((bad & lm) << len);
                            unsigned long long mh, ml, kh, kl;
                            mask_ge128(2 * (lo + len), mh, ml);
                            kh = chi & mh; kl = clo & ml;
                            unsigned long long lh, ll;
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
                    if (lane == 31) sm.cnt[c] = inc;
                    // ================= append to the chunk's slot =================================================
                    uint32_t *const cwp = stB + S0W + c * CWS;
                    uint32_t *const fwp = stB + SW8_CODE + S0W + c * FWS;
                    const uint32_t C0 = (uint32_t)(chi >> 32), C1 = (uint32_t)chi, C2 = (uint32_t)(clo >> 32), C3 = (uint32_t)clo;
                    const uint32_t bh = (uint32_t)(bad >> 32), bl = (uint32_t)bad;
                    if (wfull) {
                        reinterpret_cast<uint4 *>(cwp)[lane] = make_uint4(C0, C1, C2, C3);
                        reinterpret_cast<uint2 *>(fwp)[lane] = make_uint2(bh, bl);
                    } else if (__all_sync(FULL, n >= 32)) {
                        // every lane fills at least one whole word: each word is written once, by the lane that holds its
                        // last bits; the bits of a lane's last partial word go to the next lane by shuffle
                        const int u = inc - n;
                        {
                            const int cw0 = u >> 4, csh = 2 * (u & 15), cend = csh + 2 * n;      // cend in [64, 158]
                            const uint32_t w0 = C0 >> csh, w1 = __funnelshift_r(C1, C0, csh), w2 = __funnelshift_r(C2, C1, csh),
                                           w3 = __funnelshift_r(C3, C2, csh), w4 = __funnelshift_r(0u, C3, csh);
                            const int li = cend >> 5;                                            // 2, 3 or 4
                            uint32_t part = li == 2 ? w2 : (li == 3 ? w3 : w4);
                            if ((cend & 31) == 0) part = 0u;
                            uint32_t prev = __shfl_up_sync(FULL, part, 1);
                            if (lane == 0) prev = 0u;
                            cwp[cw0] = w0 | prev;
                            cwp[cw0 + 1] = w1;
                            if (cend >= 96) cwp[cw0 + 2] = w2;
                            if (cend >= 128) cwp[cw0 + 3] = w3;
                            if (lane == 31 && (cend & 31)) cwp[cw0 + li] = part;
                        }
                        {
                            const int fw0 = u >> 5, fsh = u & 31, fend = fsh + n;                // fend in [32, 95]
                            const uint32_t w0 = bh >> fsh, w1 = __funnelshift_r(bl, bh, fsh), w2 = __funnelshift_r(0u, bl, fsh);
                            const int li = fend >> 5;                                            // 1 or 2
                            uint32_t part = li == 1 ? w1 : w2;
                            if ((fend & 31) == 0) part = 0u;
                            uint32_t prev = __shfl_up_sync(FULL, part, 1);
                            if (lane == 0) prev = 0u;
                            fwp[fw0] = w0 | prev;
                            if (fend >= 64) fwp[fw0 + 1] = w1;
                            if (lane == 31 && (fend & 31)) fwp[fw0 + li] = part;
                        }
                    } else {
                        // some lane keeps fewer than 32 bases (header text, the end of the data): zero the slot, OR the pieces in
#pragma unroll
                        for (int i = 0; i < CWS / 32; ++i) cwp[lane + 32 * i] = 0u;
#pragma unroll
                        for (int i = 0; i < FWS / 32; ++i) fwp[lane + 32 * i] = 0u;
                        __syncwarp();
                        if (n > 0) {
                            const int u = inc - n;
                            const int cw0 = u >> 4, csh = 2 * (u & 15);
                            const int cend = csh + 2 * n;
                            uint32_t cwv[5];
                            cwv[0] = C0 >> csh;
                            cwv[1] = __funnelshift_r(C1, C0, csh);
                            cwv[2] = __funnelshift_r(C2, C1, csh);
                            cwv[3] = __funnelshift_r(C3, C2, csh);
                            cwv[4] = __funnelshift_r(0u, C3, csh);
#pragma unroll
                            for (int i = 0; i < 5; ++i)
                                if (32 * i < cend && cwv[i]) atomicOr(&cwp[cw0 + i], cwv[i]);
                            const int fw0 = u >> 5, fsh = u & 31, fend = fsh + n;
                            uint32_t bwv[3];
                            bwv[0] = bh >> fsh; bwv[1] = __funnelshift_r(bl, bh, fsh); bwv[2] = __funnelshift_r(0u, bl, fsh);
#pragma unroll
                            for (int i = 0; i < 3; ++i)
                                if (32 * i < fend && bwv[i]) atomicOr(&fwp[fw0 + i], bwv[i]);
                        }
                        __syncwarp();
                    }
                    if (e_cnt) {                                         // warp-uniform: chunk-relative kept index of the record starts
                        sm.wk[warp][lane] = keep; sm.offw[warp][lane] = (uint16_t)(inc - n);
                        __syncwarp();
                        for (int e = e_lo + lane; e < e_lo + e_cnt; e += 32) {
                            const int p = (m <= EVW ? sm.ev_p[par][e] : (int)(rec_pos(A, r_lo + e) - t0)) - cbo;
                            const int o = p >> 6, q = p & 63;
                            const int kidx = (int)sm.offw[warp][o] + (q ? __popcll(sm.wk[warp][o] >> (64 - q)) : 0);
                            if (m <= EVW) sm.ev_k[b][e] = kidx; else A.rec_k[r_lo + e] = kidx;
                        }
                        __syncwarp();
                    }
                }
                __syncthreads();                                         // ---- D: slots, counts, summaries, record-start indices
                if (!P.strip_headers || pass == 1 || !sm.assumed[par]) break;
                // ---- some chunk assumed its entry state: warp 0 composes the summaries and checks every assumption ----
                if (warp == 0) {
                    uint32_t i_hr = 0, i_x = LS_LINE_START;              // identity for lanes beyond the last chunk
                    if (lane < nch) { const uint32_t sv = sm.sum[lane]; i_hr = sv >> 2; i_x = sv & 3u; }
                    ls_scan(i_hr, i_x, lane);
                    const uint32_t u_hr = __shfl_sync(FULL, i_hr, 31), u_x = __shfl_sync(FULL, i_x, 31);   // the super-tile
                    uint32_t state = ls_known;
                    if (ls_known == LS_UNKNOWN) {
                        // entry line state of the super-tile from the chain (see encode_v5.cuh)
                        const uint32_t tagL = gen << 8;
                        if (lane == 0) st_vol32(&A.ls[tile], tagL | ((u_hr ? LK_FINAL : LK_SUMMARY) << 2) | u_x);
                        bool ok = true;
                        uint32_t carry = LS_LINE_START; bool have_carry = false;
                        for (int bs = tile - 1;; bs -= 32) {             // tile > 0: tile 0's entry state is always known
                            const int j = bs - lane;
                            uint32_t kind = LK_FINAL, val = LS_LINE_START;
                            int f = 32;
                            for (int spins = 0;; ++spins) {
                                if (j >= 0) {
                                    const uint32_t a = ld_vol32(&A.ls[j]);
                                    kind = (a >> 8) == (gen & 0xffffffu) ? ((a >> 2) & 3u) : LK_NONE;
                                    val = a & 3u;
                                }
                                const uint32_t tb = __ballot_sync(FULL, kind == LK_FINAL);
                                f = tb ? __ffs(tb) - 1 : 32;
                                const uint32_t missing = __ballot_sync(FULL, kind == LK_NONE) & (f < 32 ? ((1u << f) - 1u) : FULL);
                                if (!missing) break;
                                if (spins > SPIN_LIMIT) { ok = false; break; }
                                __nanosleep(40);
                            }
                            if (!ok) break;
                            const uint32_t nb = __ballot_sync(FULL, val != LS_LINE_START && lane <= f);
                            if (nb) { carry = __shfl_sync(FULL, val, 31 - __clz(nb)); have_carry = true; }
                            if (f < 32) break;
                        }
                        state = have_carry ? carry : LS_LINE_START;
                        if (!ok && lane == 0) A.status[1] = 1u;
                        if (lane == 0) st_vol32(&A.ls[tile], tagL | (LK_FINAL << 2) | ls_apply(u_hr, u_x, state));
                    }
                    uint32_t e_hr = __shfl_up_sync(FULL, i_hr, 1), e_x = __shfl_up_sync(FULL, i_x, 1);
                    if (lane == 0) { e_hr = 0; e_x = LS_LINE_START; }
                    const uint32_t et = ls_apply(e_hr, e_x, state);      // true entry state of chunk `lane`
                    const bool wrong = lane < nch && et != (uint32_t)sm.ent_used[lane];
                    if (lane < nch) sm.ent_true[lane] = (uint8_t)et;
                    const uint32_t anyw = __ballot_sync(FULL, wrong);
                    if (lane == 0) sm.redo = anyw != 0u;
                }
                __syncthreads();                                         // ---- true entry states
                if (!sm.redo) break;
            }
            if (m > EVW) {
                // many record starts: their chunk-relative kept indices (rec_k) become super-tile-relative
                const int cn = lane < nch ? sm.cnt[lane] : 0;
                int inc = cn;
#pragma unroll
                for (int d = 1; d < 32; d <<= 1) { const int t = __shfl_up_sync(FULL, inc, d); if (lane >= d) inc += t; }
                const int exc = inc - cn;
                // every warp writes the same prefix values: shared memory serves the look-up by chunk
                sm.pre[b][1 + lane] = PEND + exc;
                __syncwarp();
                for (int e = tid; e < m; e += NT) {
                    const int ch = (int)((rec_pos(A, r_lo + e) - t0) >> 11);
                    const int add = sm.pre[b][1 + ch] - PEND;
                    if (add) __stcg(A.rec_k + r_lo + e, __ldcg(A.rec_k + r_lo + e) + add);
                }
                __syncthreads();
            }
        } else {
            __syncthreads();                                             // ---- D
        }

        // ================= warp NW-1: next ticket; warp 1: aggregate(B); warp 0: look-back(A) ======================
        if (warp == NW - 1) {
            if (haveB) {
                next_ticket = __shfl_sync(FULL, next_ticket, 0);
                prep_super(A, sm, par ^ 1, next_ticket, lane, pos_first, pos_last);
            } else if (lane == 0) {
                sm.c_tile[par ^ 1] = A.n_tiles;
            }
            if (lane == 0) sm.assumed[par ^ 1] = 0u;
        }
        const uint32_t tagA = (gen << 2) | ST_AGG, tagI = (gen << 2) | ST_INCL;
        if (warp == 1 || warp == 0) {
            if (warp == 1 && haveB) {
                // ---- slot prefix, aggregate of super-tile B and the segment table of its record starts ----------------
                const int cn = lane < nch ? sm.cnt[lane] : 0;
                int cinc = cn;
#pragma unroll
                for (int d = 1; d < 32; d <<= 1) { const int t = __shfl_up_sync(FULL, cinc, d); if (lane >= d) cinc += t; }
                const int exc = cinc - cn;
                const int ktot = __shfl_sync(FULL, cinc, 31);
                sm.pre[b][1 + lane] = PEND + exc;
                if (lane == 0) { sm.pre[b][0] = 0; sm.pre[b][NCH + 1] = PEND + ktot; }
                __syncwarp();
                const Strm ZB{stB, sm.pre[b]};
                int fk, lk, closed = 0, ntok = 0;
                if (m == 0) { fk = ktot; lk = ktot; }
                else if (m <= EVW) {
                    const int ech = lane < m ? (sm.ev_p[par][lane] >> 11) : 0;
                    const int eb = __shfl_sync(FULL, exc, ech);
                    const int ke = lane < m ? sm.ev_k[b][lane] + eb : ktot;
                    int kn = __shfl_down_sync(FULL, ke, 1);
                    if (lane >= m - 1) kn = ktot;
                    const int ne = kn - ke;
                    const int nw = (int)div_k((uint32_t)ne, P);
                    const int te = lane < m - 1 ? nw + tail_tokens(ne - nw * k, P) : (lane == m - 1 ? nw : 0);
                    int ti = te;
#pragma unroll
                    for (int d = 1; d < 32; d <<= 1) { const int t = __shfl_up_sync(FULL, ti, d); if (lane >= d) ti += t; }
                    const int ex = ti - te;
                    ntok = __shfl_sync(FULL, ti, 31); closed = __shfl_sync(FULL, ex, m - 1);
                    if (lane < m) { sm.seg_src[b][1 + lane] = PEND + ke; sm.seg_t[b][1 + lane] = ex; sm.seg_nwin[b][1 + lane] = nw; }
                    fk = __shfl_sync(FULL, ke, 0); lk = __shfl_sync(FULL, ne, m - 1);
                } else {
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
                const int tn = min(k - 1, lk);
                unsigned long long gtail = 0;
                {
                    unsigned long long tl = 0;
                    if (lane < tn) tl = (unsigned long long)class_at8(ZB, PEND + ktot - tn + lane) << (3 * (tn - 1 - lane));
                    gtail = ((unsigned long long)__reduce_or_sync(FULL, (uint32_t)(tl >> 32)) << 32) | __reduce_or_sync(FULL, (uint32_t)tl);
                }
                // line-state word of a super-tile whose entry state was known up front
                uint32_t u_hr = 0, u_x = LS_LINE_START;
                const bool pub_ls = P.strip_headers && sm.c_ls[par] != LS_UNKNOWN;
                if (pub_ls) {
                    if (lane < nch) { const uint32_t sv = sm.sum[lane]; u_hr = sv >> 2; u_x = sv & 3u; }
                    ls_scan(u_hr, u_x, lane);
                    u_hr = __shfl_sync(FULL, u_hr, 31); u_x = __shfl_sync(FULL, u_x, 31);
                }
                if (lane == 0) {
                    TileDesc &D = A.descs[tile];
                    st_vol128(&D.a0, make_uint4(tagA, (uint32_t)fk, (uint32_t)lk, (uint32_t)closed | ((uint32_t)(m > 0) << 31)));
                    st_vol128(&D.a1, make_uint4(tagA, (uint32_t)tn | ((uint32_t)(gtail >> 32) << 4), (uint32_t)gtail, 0u));
                    TileAgg &g = sm.ag[b];
                    g.fk = fk; g.lk = lk; g.closed = closed; g.tn = tn; g.ntok = ntok; g.hasev = m > 0; g.tail = gtail;
                    if (pub_ls) st_vol32(&A.ls[tile], (gen << 8) | (LK_FINAL << 2) | ls_apply(u_hr, u_x, sm.c_ls[par]));
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
                // carried bases of the open record: slot 0, right-aligned in front of position PEND
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
                    if (lane == 0) { stA[0] = cw; stA[1] = 0u; stA[SW8_CODE] = fw; stA[SW8_CODE + 1] = 0u; }
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
            const Strm ZA{sm.strm[ba], sm.pre[ba]};
            const int ktotA = sm.pre[ba][NCH + 1] - PEND;
            const int64_t T0 = sm.T0;
            const int a = (int)(T0 & (R - 1));
            const int64_t gbase = T0 - a;
            const int64_t capl = A.ids_cap - gbase;
            const int cap_rel = capl < 0 ? 0 : (capl > 0x7fffffff ? 0x7fffffff : (int)capl);
            const int tok0 = sm.tok0;
            if (mA <= EVW) {
                SegTab G; G.src = sm.seg_src[ba]; G.t = sm.seg_t[ba]; G.nwin = sm.seg_nwin[ba];
                if (tid < mA) A.out_off[rloA + tid] = T0 + G.t[1 + tid];
                emit_segments8<IdT, KK>(A, ZA, G, mA + 1, sm.ntok, a, gbase, cap_rel, vec_ok, affine);
            } else {
                SegTab G; G.src = sm.ent_src; G.t = sm.ent_t; G.nwin = sm.ent_nwin;
                if (tid == 0) { sm.ent_src[0] = sm.seg_src[ba][0]; sm.ent_t[0] = 0; sm.ent_nwin[0] = sm.seg_nwin[ba][0]; }
                int tbase = tok0;
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
                    emit_range8<IdT, KK>(A, ZA, G, c0 == 0 ? 0 : tbase, tbase + total, cm + 1, a, gbase, cap_rel, vec_ok, affine);
                    tbase += total;
                    __syncthreads();
                }
            }
        }
        __syncthreads();                                         // ---- A's buffer and tables are free again
        haveA = haveB; tileA = tile; mA = m; rloA = r_lo; b ^= 1;
    }
}

}  // namespace v8
}  // namespace dtk
