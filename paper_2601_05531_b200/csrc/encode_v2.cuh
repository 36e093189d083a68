// encode_v2.cuh -- single-pass classify + strip + {single-nt | k-mer} + CSR offsets, bit-plane form.
//
// One persistent CTA (256 threads) claims flat 16 KiB byte tiles in order (atomic ticket); each thread owns
// 64 contiguous input bytes, loaded straight into registers with four 16-byte loads.  Per tile:
//   1. classify ("256-entry LUT"; Alg. 1): ACGT in either case is recognised
//      arithmetically on four bytes per 32-bit register -- the 2-bit code is ASCII bits 1..2, validity is one
//      masked compare -- and gathered into per-thread bit planes by a multiply (code plane: 2 bits x 64
//      bases, exception plane: 1 bit x 64).  Every byte the arithmetic does not prove to be ACGT (newlines,
//      N, '>', IUPAC codes, anything a custom table redefines) is classified through the 256-entry LUT in
//      shared memory, one byte at a time: the table remains the specification.  A table that disagrees with the
//      default on ACGTacgt sends every byte through the LUT.
//   2. line state (LINE_START / IN_LINE / IN_HEADER) per thread as a 3-bit function summary, composed by a
//      warp shuffle scan, across warps through shared memory and across tiles by a look-back chain of its own
//   3. keep = in-record & ~SKIP & ~header; the planes are compacted in registers by deleting dropped bits,
//      a block prefix scan of popc(keep) gives each thread's position in the tile's kept-base stream, and the
//      planes are appended to that stream in shared memory (2-bit base-4 digits, most significant first)
//   4. tile aggregate published; warp-parallel decoupled look-back gives the inclusive prefix (out_offsets of
//      the open record, its kept-base count, its pending partial window)
//   5. tokens are cut from the stream per record segment in groups of 16 output bytes: one funnel-shift
//      alignment per group, windows at compile-time offsets, one 16-byte store straight to ids_out.
// Input bytes are read from HBM exactly once and ids written exactly once.
#pragma once
#include "common.cuh"

namespace dtk {

constexpr int LB = 64;                       // bytes per thread
constexpr int TB2 = NT * LB;                 // tile bytes (16 KiB)
constexpr int NW = NT / 32;
constexpr int PEND = 16;                     // stream slots in front of the tile's kept bases (carried bases)
constexpr int SW_CODE = (PEND + TB2) / 16 + 8;
constexpr int SW_FLAG = (PEND + TB2) / 32 + 8;
constexpr int EV_CAP = NT;                   // record starts handled per pass of the event loop

struct Smem2 {
    uint32_t cs[SW_CODE];                    // code stream: base u at word u>>4, bits 31-2(u&15) .. 30-2(u&15)
    uint32_t bs[SW_FLAG];                    // "not ACGT" stream: base u at word u>>5, bit 31-(u&31)
    uint32_t ns[SW_FLAG];                    // "is N" stream (subset of bs)
    unsigned long long keep[NT];             // keep mask per thread, byte q at bit 63-q
    unsigned long long rs[NT];               // record starts per thread, same bit order
    int32_t scan[NT];                        // exclusive kept-base prefix per thread
    int32_t ev_k[EV_CAP], ev_n[EV_CAP];
    long long ev_out[EV_CAP];
    int32_t warp_tmp[NW];
    uint32_t warp_ls[NW];
    uint8_t lut[256];
    int32_t tile, ktot, any_rs;
    long long r_lo, r_hi;
    uint32_t ls_in;
    Prefix pin;
};

// ---------------------------------------------------------------------------------------- small helpers
__device__ __forceinline__ unsigned long long bit_at(int q) { return 1ull << (63 - q); }          // q in 0..63
__device__ __forceinline__ unsigned long long from_pos(int q) { return q >= 64 ? 0ull : (~0ull >> q); }   // positions >= q
__device__ __forceinline__ int first_pos(unsigned long long m) { return m ? __clzll((long long)m) : 64; }
__device__ __forceinline__ int last_pos(unsigned long long m) { return 63 - (__ffsll((long long)m) - 1); }   // m != 0

// exclusive block scan of one int per thread (two barriers)
__device__ __forceinline__ int block_exscan2(int v, Smem2 &sm, int &total) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    int inc = v;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) { int t = __shfl_up_sync(0xffffffffu, inc, d); if (lane >= d) inc += t; }
    if (lane == 31) sm.warp_tmp[warp] = inc;
    __syncthreads();
    int woff = 0, tot = 0;
#pragma unroll
    for (int w = 0; w < NW; ++w) { int t = sm.warp_tmp[w]; if (w < warp) woff += t; tot += t; }
    __syncthreads();
    total = tot;
    return woff + inc - v;
}

__device__ __forceinline__ int64_t rec_pos2(const EncArgs &A, int64_t r) { return A.rec_off[r] - A.off_bias + A.mis; }

// first r in [lo, n_rec + 1) with rec_pos(r) >= pos; warp-cooperative 32-ary search (all lanes return it)
__device__ __forceinline__ int64_t warp_lower_bound2(const EncArgs &A, int64_t lo, int64_t pos) {
    const int lane = threadIdx.x & 31;
    int64_t hi = A.n_rec + 1;
    while (hi - lo > 32) {
        int64_t step = (hi - lo + 31) / 32;
        int64_t idx = lo + (int64_t)(lane + 1) * step - 1;
        bool ge = (idx >= hi) ? true : (rec_pos2(A, idx) >= pos);
        uint32_t b = __ballot_sync(0xffffffffu, ge);
        if (!b) return hi;
        int f = __ffs(b) - 1;
        int64_t nlo = lo + (int64_t)f * step;
        int64_t nhi = lo + (int64_t)(f + 1) * step - 1;
        if (nhi > hi) nhi = hi;
        lo = nlo; hi = nhi;
    }
    int64_t idx = lo + lane;
    bool ge = (idx >= hi) ? true : (rec_pos2(A, idx) >= pos);
    uint32_t b = __ballot_sync(0xffffffffu, ge);
    return b ? lo + (__ffs(b) - 1) : hi;
}

__device__ __forceinline__ int kept_before2(const Smem2 &sm, int p) {      // kept bases at tile positions < p
    if (p >= TB2) return sm.ktot;
    const int t = p >> 6, q = p & 63;
    return sm.scan[t] + (q ? __popcll(sm.keep[t] >> (64 - q)) : 0);
}

// ---- stream readers (dynamic position) -------------------------------------------------------------
__device__ __forceinline__ uint32_t code_at(const Smem2 &sm, int u, int k) {        // k digits starting at base u
    const int b = 2 * u, w = b >> 5, s = b & 31;
    return __funnelshift_l(sm.cs[w + 1], sm.cs[w], s) >> (32 - 2 * k);
}
__device__ __forceinline__ uint32_t flags_at(const uint32_t *st, int u, int k) {    // k flag bits starting at base u
    const int w = u >> 5, s = u & 31;
    return __funnelshift_l(st[w + 1], st[w], s) >> (32 - k);
}
__device__ __forceinline__ uint32_t class_at(const Smem2 &sm, int u) {              // class code 0..5 of base u
    if (flags_at(sm.bs, u, 1)) return flags_at(sm.ns, u, 1) ? CLS_N : CLS_UNK;
    return code_at(sm, u, 1);
}

template <typename IdT>
__device__ __forceinline__ void store_id2(const EncArgs &A, int64_t idx, int32_t id) {
    if (idx < A.ids_cap) reinterpret_cast<IdT *>(A.ids)[idx] = (IdT)id;
    else A.status[0] = 1u;
}

__device__ __forceinline__ int32_t nt_id_of(const EncParams &P, uint32_t cls) {
    return cls <= CLS_N ? P.nt_ids[cls] : P.unk_id;
}

// ---- emission ---------------------------------------------------------------------------------------
// One group = R = 16 / sizeof(IdT) consecutive output slots, aligned to 16 bytes in ids_out.  A thread that
// owns a full group inside one segment reads the stream words once, aligns them with one funnel shift per
// word and cuts R windows at compile-time offsets; partial groups fall back to one token at a time.
template <typename IdT, int K, bool SINGLE>
__device__ __forceinline__ void emit_group_fast(const EncArgs &A, const Smem2 &sm, int u, int64_t o) {
    constexpr int R = 16 / (int)sizeof(IdT);
    constexpr int CB = 2 * K * R;                        // code bits per group
    constexpr int NCW = (CB + 30) / 32 + 1;              // stream words that can be touched
    constexpr int FB = K * R;
    constexpr int NFW = (FB + 31) / 32 + 1;
    const EncParams &P = A.prm;
    uint32_t a[NCW];
    {
        const int b = 2 * u, w = b >> 5, s = b & 31;
        uint32_t raw[NCW + 1];
#pragma unroll
        for (int i = 0; i <= NCW; ++i) raw[i] = sm.cs[w + i];
#pragma unroll
        for (int i = 0; i < NCW; ++i) a[i] = __funnelshift_l(raw[i + 1], raw[i], s);
    }
    uint32_t f[NFW];
    uint32_t anybad = 0;
    {
        const int w = u >> 5, s = u & 31;
        uint32_t raw[NFW + 1];
#pragma unroll
        for (int i = 0; i <= NFW; ++i) raw[i] = sm.bs[w + i];
#pragma unroll
        for (int i = 0; i < NFW; ++i) f[i] = __funnelshift_l(raw[i + 1], raw[i], s);
#pragma unroll
        for (int i = 0; i < NFW; ++i) {
            const int lo = i * 32, hi = lo + 32;         // flag bits [lo, hi) of the group live in f[i]
            if (lo < FB) anybad |= (hi <= FB) ? f[i] : (f[i] & ~(0xffffffffu >> (FB - lo)));
        }
    }
    int32_t id[R];
#pragma unroll
    for (int t = 0; t < R; ++t) {
        constexpr int W = 2 * K;
        const int bo = W * t, i = bo >> 5, s = bo & 31;
        uint32_t c = (s + W <= 32) ? ((a[i] >> (32 - s - W)) & ((W == 32) ? 0xffffffffu : ((1u << W) - 1u)))
                                   : (__funnelshift_l(a[i + 1], a[i], s) >> (32 - W));
        id[t] = SINGLE ? (int32_t)c : (int32_t)(P.base_id + c);
    }
    if (SINGLE) {
        const bool affine = P.nt_ids[1] == P.nt_ids[0] + 1 && P.nt_ids[2] == P.nt_ids[0] + 2 && P.nt_ids[3] == P.nt_ids[0] + 3;
#pragma unroll
        for (int t = 0; t < R; ++t) id[t] = affine ? P.nt_ids[0] + id[t] : P.nt_ids[id[t]];
    }
    if (anybad) {
        uint32_t nf[NFW];
        if (SINGLE) {
            const int w = u >> 5, s = u & 31;
#pragma unroll
            for (int i = 0; i < NFW; ++i) nf[i] = __funnelshift_l(sm.ns[w + i + 1], sm.ns[w + i], s);
        }
#pragma unroll
        for (int t = 0; t < R; ++t) {
            const int bo = K * t, i = bo >> 5, s = bo & 31;
            uint32_t m = (s + K <= 32) ? ((f[i] >> (32 - s - K)) & ((1u << K) - 1u))
                                       : (__funnelshift_l(f[i + 1], f[i], s) >> (32 - K));
            if (m) id[t] = (SINGLE && ((nf[i] >> (31 - s)) & 1u)) ? P.nt_ids[4] : P.unk_id;
        }
    }
    IdT *dst = reinterpret_cast<IdT *>(A.ids) + o;
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

// one token, any k (dynamic shifts)
template <typename IdT>
__device__ __forceinline__ void emit_token_slow(const EncArgs &A, const Smem2 &sm, int u, int64_t o) {
    const EncParams &P = A.prm;
    int32_t id;
    if (P.mode == MODE_KMER) {
        id = flags_at(sm.bs, u, P.k) ? P.unk_id : (int32_t)(P.base_id + code_at(sm, u, P.k));
    } else {
        id = nt_id_of(P, class_at(sm, u));
    }
    store_id2<IdT>(A, o, id);
}

// tokens [0, nwin) of a segment whose first window starts at stream base u0; token j goes to ids[out_base + j].
// g / gs: index within / size of the cooperating thread group.
template <typename IdT, int K, bool SINGLE>
__device__ __forceinline__ void emit_windows(const EncArgs &A, const Smem2 &sm, int u0, int nwin, int64_t out_base,
                                             int g, int gs) {
    constexpr int R = 16 / (int)sizeof(IdT);
    const int kk = SINGLE ? 1 : (K > 0 ? K : A.prm.k);
    if (nwin <= 0) return;
    const int64_t o_end = out_base + nwin;
    const int64_t g_first = out_base / R;                // aligned groups covering [out_base, o_end)
    const int n_groups = (int)((o_end + R - 1) / R - g_first);
    for (int q = g; q < n_groups; q += gs) {
        const int64_t o0 = (g_first + q) * R;
        const int64_t lo = o0 < out_base ? out_base : o0, hi = (o0 + R < o_end) ? o0 + R : o_end;
        if (K > 0 && lo == o0 && hi == o0 + R && o0 + R <= A.ids_cap && (reinterpret_cast<uintptr_t>(A.ids) & 15) == 0) {
            emit_group_fast<IdT, (K > 0 ? K : 1), SINGLE>(A, sm, u0 + (int)(o0 - out_base) * kk, o0);
        } else {
            for (int64_t o = lo; o < hi; ++o) emit_token_slow<IdT>(A, sm, u0 + (int)(o - out_base) * kk, o);
        }
    }
}

// emit the tokens of one record piece: `n` bases available from stream base `src` (carried bases included);
// `closes`: the record ends inside this tile, so the n mod k trailing bases are emitted under the tail policy.
template <typename IdT>
__device__ __forceinline__ void emit_segment2(const EncArgs &A, const Smem2 &sm, int src, int n, bool closes,
                                              int64_t out_base, int g, int gs) {
    const EncParams &P = A.prm;
    if (P.mode != MODE_KMER) {
        emit_windows<IdT, 1, true>(A, sm, src, n, out_base, g, gs);
        return;
    }
    const int k = P.k, nwin = n / k, rem = n - nwin * k;
    switch (k) {
        case 1: emit_windows<IdT, 1, false>(A, sm, src, nwin, out_base, g, gs); break;
        case 2: emit_windows<IdT, 2, false>(A, sm, src, nwin, out_base, g, gs); break;
        case 3: emit_windows<IdT, 3, false>(A, sm, src, nwin, out_base, g, gs); break;
        case 4: emit_windows<IdT, 4, false>(A, sm, src, nwin, out_base, g, gs); break;
        case 5: emit_windows<IdT, 5, false>(A, sm, src, nwin, out_base, g, gs); break;
        case 6: emit_windows<IdT, 6, false>(A, sm, src, nwin, out_base, g, gs); break;
        case 8: emit_windows<IdT, 8, false>(A, sm, src, nwin, out_base, g, gs); break;
        default: emit_windows<IdT, 0, false>(A, sm, src, nwin, out_base, g, gs); break;
    }
    if (closes && rem) {
        if (P.tail_policy == TAIL_PER_BASE) {
            for (int i = g; i < rem; i += gs) {
                uint32_t ci = class_at(sm, src + nwin * k + i);
                store_id2<IdT>(A, out_base + nwin + i, ci <= CLS_N ? (int32_t)(P.base_id + P.four_k + ci) : P.unk_id);
            }
        } else if (P.tail_policy == TAIL_UNK) {
            if (g == 0) store_id2<IdT>(A, out_base + nwin, P.unk_id);
        }
    }
}

// ---- classification -----------------------------------------------------------------------------------
// Four bytes per register.  Returns through `code` the raw 2-bit codes (ASCII bits 1..2: A 00, C 01, G 11,
// T 10) of bytes 0..3 in bits 24..31 (byte 0 lowest) and through `flag` 0x80 in every byte that is not one of
// ACGTacgt.  valid <=> (x & 0xD9) == (T-pattern ? 0x50 : 0x41), T-pattern <=> bits(2,1) == (1,0).
__device__ __forceinline__ void classify_word(uint32_t x, uint32_t &code, uint32_t &flag) {
    code = (x & 0x06060606u) * 0x00820820u;
    const uint32_t m = (x >> 2) & ~(x >> 1) & 0x01010101u;           // 1 where the byte has the T pattern
    const uint32_t d = ((x & 0x59595959u) ^ 0x41414141u) ^ (m * 0x11u); // 0 <=> valid (0x41 ^ 0x11 = 0x50 for T)
    const uint32_t a = d + 0x7f7f7f7fu;                              // bit 7 of each byte <=> byte of d non-zero (d < 0x80)
    flag = (a | x) & 0x80808080u;                                    // bytes >= 0x80 are never DNA
}

template <typename IdT>
__global__ void __launch_bounds__(NT) encode_tiles_v2(const __grid_constant__ EncArgs A) {
    extern __shared__ __align__(16) uint8_t smem_raw[];
    Smem2 &sm = *reinterpret_cast<Smem2 *>(smem_raw);
    const EncParams &P = A.prm;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const uint32_t gen = A.gen;
    const bool need_n = (P.mode != MODE_KMER) || (P.tail_policy == TAIL_PER_BASE);

    sm.lut[tid] = A.lut[tid];
    const int64_t pos_first = rec_pos2(A, 0), pos_last = rec_pos2(A, A.n_rec);   // bytes outside are in no record

    for (;;) {
        __syncthreads();
        if (tid == 0) {
            sm.tile = (int)(atomicAdd(A.ticket, 1ull) - A.ticket_base);
            sm.bs[0] = 0; sm.ns[0] = 0; sm.any_rs = 0;
        }
        sm.rs[tid] = 0ull;
        __syncthreads();
        const int tile = sm.tile;
        if (tile >= A.n_tiles) break;
        const int64_t t0 = (int64_t)tile * TB2;
        const int64_t p0 = t0 + (int64_t)tid * LB;             // position of this thread's first byte
        TileDesc &D = A.descs[tile];

        // ---- 1. load: 4 x 16 bytes per thread -------------------------------------------------------
        uint4 v[4];
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const int64_t p = p0 + 16 * j;
            v[j] = (p < A.p_end) ? __ldg(reinterpret_cast<const uint4 *>(A.bytes_al + p)) : make_uint4(0, 0, 0, 0);
        }
        // ---- record starts inside the tile (warp 0, while the loads are in flight) -------------------
        if (warp == 0) {
            int64_t rlo = warp_lower_bound2(A, 0, t0);
            int64_t rhi = (tile == A.n_tiles - 1) ? A.n_rec + 1 : warp_lower_bound2(A, rlo, t0 + TB2);
            if (lane == 0) { sm.r_lo = rlo; sm.r_hi = rhi; sm.any_rs = rhi > rlo; }
            for (int64_t e = rlo + lane; e < rhi; e += 32) {
                int p = (int)(rec_pos2(A, e) - t0);
                atomicOr(&sm.rs[p >> 6], bit_at(p & 63));
            }
        }

        // ---- 2. classify ---------------------------------------------------------------------------------
        uint32_t C[4];                                      // code plane, MSB first, 16 bases per word
        unsigned long long E;                               // exception plane: not provably ACGT
        {
            const uint32_t *xw = reinterpret_cast<const uint32_t *>(v);
            uint32_t cb[16], fb[16];
#pragma unroll
            for (int j = 0; j < 16; ++j) classify_word(xw[j], cb[j], fb[j]);
            uint32_t el[2];
#pragma unroll
            for (int h = 0; h < 4; ++h) {
                // codes: top bytes of four products -> one LSB-first word of 16 bases -> MSB first, Gray -> binary
                uint32_t lo2 = __byte_perm(cb[4 * h], cb[4 * h + 1], 0x0073);      // bytes: [p0.3, p1.3, 0, 0]
                uint32_t hi2 = __byte_perm(cb[4 * h + 2], cb[4 * h + 3], 0x0073);
                uint32_t wl = __byte_perm(lo2, hi2, 0x5410);                        // [lo2.0, lo2.1, hi2.0, hi2.1]
                uint32_t y = __brev(wl);                     // base 0 now in bits 31..30 with its two bits swapped
                // field holds (lo, hi) of the Gray code (hi = ASCII bit 2, lo = ASCII bit 1): binary = (hi, lo ^ hi)
                C[h] = ((y & 0x55555555u) << 1) | (((y >> 1) ^ y) & 0x55555555u);
            }
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                uint32_t b[4];
#pragma unroll
                for (int pr = 0; pr < 4; ++pr) {
                    // two words -> one byte: flags of the even word in the low nibble, of the odd word in the high one
                    uint32_t fa = fb[8 * h + 2 * pr + 1] | (fb[8 * h + 2 * pr] >> 4);
                    b[pr] = fa * 0x00204081u;                // byte at bits 24..31, first input byte lowest
                }
                uint32_t lo2 = __byte_perm(b[0], b[1], 0x0073), hi2 = __byte_perm(b[2], b[3], 0x0073);
                el[h] = __brev(__byte_perm(lo2, hi2, 0x5410));
            }
            E = ((unsigned long long)el[0] << 32) | el[1];
        }
        if (!P.fast_lut) E = ~0ull;

        // ---- exceptions through the 256-entry LUT -----------------------------------------------------------
        unsigned long long skip = 0, nl = 0, gt = 0, nm = 0, bad = E;
        {
            const uint8_t *vb = reinterpret_cast<const uint8_t *>(A.bytes_al) + p0;
            unsigned long long rem = E;
            while (rem) {
                const int q = __clzll((long long)rem);
                const unsigned long long bq = bit_at(q);
                rem &= ~bq;
                const uint32_t byte = (p0 + q < A.p_end) ? (uint32_t)__ldg(vb + q) : 0u;
                const uint32_t c = sm.lut[byte];
                if (c == CLS_SKIP) { skip |= bq; bad &= ~bq; if (byte == '\n') nl |= bq; }
                else if (c == CLS_N) nm |= bq;
                else if (c < CLS_N) {                        // a table entry that maps this byte to a base
                    bad &= ~bq;
                    const int sh = 30 - 2 * (q & 15);
                    const uint32_t msk = ~(3u << sh), val = c << sh;
                    switch (q >> 4) {
                        case 0: C[0] = (C[0] & msk) | val; break;
                        case 1: C[1] = (C[1] & msk) | val; break;
                        case 2: C[2] = (C[2] & msk) | val; break;
                        default: C[3] = (C[3] & msk) | val; break;
                    }
                }
                if (byte == '>') gt |= bq;
            }
        }
        __syncthreads();                                     // record-start bitmap complete
        const unsigned long long rs = sm.any_rs ? sm.rs[tid] : 0ull;
        const int64_t r_lo = sm.r_lo;
        const int m = (int)(sm.r_hi - r_lo);                 // events in this tile

        // ---- 3. line state + header lines --------------------------------------------------------------------
        unsigned long long hdr = 0;
        if (P.strip_headers) {
            const unsigned long long osk = skip & ~nl;
            // line starts: after each '\n', at each record start, and (hypothetically) at the thread's first byte
            auto settle = [&](unsigned long long ls, bool &pending) {   // move line starts over non-newline SKIP bytes
                pending = (nl & 1ull) != 0;
                unsigned long long t;
                while ((t = ls & osk) != 0) { pending = pending || (t & 1ull); ls = (ls & ~t) | (t >> 1); }
                return ls;
            };
            auto exit_state = [&](unsigned long long ls, bool pending, uint32_t entry) -> uint32_t {
                if (pending) return LS_LINE_START;
                if (!ls) return entry;
                const unsigned long long lastb = ls & (~ls + 1ull);      // lowest set bit = last line start
                return (gt & lastb) ? LS_IN_HEADER : LS_IN_LINE;
            };
            const unsigned long long ls_base = (nl >> 1) | rs;
            const bool has_reset = (nl | rs) != 0;
            bool pend0;
            const unsigned long long ls0 = settle(ls_base | bit_at(0), pend0);
            const uint32_t x = exit_state(ls0, pend0, LS_LINE_START);
            // inclusive warp scan of (has_reset, x) under composition
            uint32_t s_hr = has_reset, s_x = x;
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) {
                uint32_t o_hr = __shfl_up_sync(0xffffffffu, s_hr, d), o_x = __shfl_up_sync(0xffffffffu, s_x, d);
                if (lane >= d) {                             // (earlier o) then (later s)
                    s_x = s_hr ? s_x : (o_x == LS_LINE_START ? s_x : o_x);
                    s_hr |= o_hr;
                }
            }
            if (lane == 31) sm.warp_ls[warp] = (s_hr << 2) | s_x;
            uint32_t e_hr = __shfl_up_sync(0xffffffffu, s_hr, 1), e_x = __shfl_up_sync(0xffffffffu, s_x, 1);
            if (lane == 0) { e_hr = 0; e_x = LS_LINE_START; }          // identity: f(e) = e (x = LINE_START, no reset)
            __syncthreads();
            if (tid == 0) {
                uint32_t t_hr = 0, t_x = LS_LINE_START;
                for (int w = 0; w < NW; ++w) {
                    uint32_t v2 = sm.warp_ls[w], g_hr = v2 >> 2, g_x = v2 & 3u;
                    t_x = g_hr ? g_x : (t_x == LS_LINE_START ? g_x : t_x);
                    t_hr |= g_hr;
                }
                st_vol32(&D.l_word, (gen << 8) | (t_hr << 2) | t_x);
                sm.ls_in = (t_hr << 2) | t_x;                // parked for warp 0 below
            }
            __syncthreads();
            if (warp == 0) {
                // entry state of the tile: nearest predecessor whose exit state is known, then the x of every
                // tile in between applies only while the state is still LINE_START
                const uint32_t mine = sm.ls_in;
                uint32_t state = LS_LINE_START;
                bool found = (tile == 0), ok = true;
                uint32_t carry = LS_LINE_START;              // first non-LINE_START x among nearer tiles already scanned
                bool have_carry = false;
                for (int base = tile - 1; !found && ok; base -= 32) {
                    const int j = base - lane;
                    uint32_t val = LS_LINE_START; bool term = true;      // tiles before 0: known LINE_START
                    if (j >= 0) {
                        const TileDesc &Dj = A.descs[j];
                        int spins = 0;
                        for (;;) {
                            uint32_t a = ld_vol32(&Dj.l_incl);
                            if ((a >> 8) == gen) { val = a & 3u; term = true; break; }
                            a = ld_vol32(&Dj.l_word);
                            if ((a >> 8) == gen) { val = a & 3u; term = (a >> 2) & 1u; break; }
                            if (++spins > SPIN_LIMIT) { ok = false; break; }
                        }
                    }
                    ok = __all_sync(0xffffffffu, ok);
                    if (!ok) break;
                    const uint32_t tb = __ballot_sync(0xffffffffu, term);
                    const int f = tb ? __ffs(tb) - 1 : 32;                 // nearest terminal lane
                    // candidates: lanes <= f (nearer tiles have lower lanes); the value that survives is the one of the
                    // farthest lane <= f whose value is not LINE_START
                    const uint32_t nb = __ballot_sync(0xffffffffu, val != LS_LINE_START && lane <= f);
                    if (nb) {                                // a farther non-LINE_START value overrides nearer ones
                        carry = __shfl_sync(0xffffffffu, val, 31 - __clz(nb));
                        have_carry = true;
                    }
                    found = f < 32;
                }
                // `carry` holds the farthest non-LINE_START value seen up to the terminal tile
                state = have_carry ? carry : LS_LINE_START;
                if (!ok) { if (lane == 0) A.status[1] = 1u; }
                if (lane == 0) {
                    const uint32_t t_hr = mine >> 2, t_x = mine & 3u;
                    const uint32_t ex = t_hr ? t_x : (state == LS_LINE_START ? t_x : state);
                    st_vol32(&D.l_incl, (gen << 8) | ex);
                    sm.ls_in = state;
                }
            }
            __syncthreads();
            // entry state of this thread
            uint32_t st_in = sm.ls_in;
            for (int w = 0; w < warp; ++w) {
                uint32_t v2 = sm.warp_ls[w], g_hr = v2 >> 2, g_x = v2 & 3u;
                st_in = g_hr ? g_x : (st_in == LS_LINE_START ? g_x : st_in);
            }
            st_in = e_hr ? e_x : (st_in == LS_LINE_START ? e_x : st_in);
            // header bytes
            bool pd;
            unsigned long long ls = settle(ls_base | (st_in == LS_LINE_START ? bit_at(0) : 0ull), pd);
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

        // ---- 4. keep mask, in-register compaction, block scan, stream append ------------------------------------
        unsigned long long keep = ~skip & ~hdr;
        {
            const int64_t a = pos_first - p0, b = pos_last - p0;        // in-record positions are [a, b)
            const unsigned long long ma = a <= 0 ? ~0ull : from_pos((int)(a > 64 ? 64 : a));
            const unsigned long long mb = b <= 0 ? 0ull : (b >= 64 ? ~0ull : ~from_pos((int)b));
            keep &= ma & mb;
        }
        const int n = __popcll(keep);
        if (keep != ~0ull) {
            // delete the dropped positions from the planes, highest position first so lower ones stay valid
            unsigned long long drop = ~keep;
            if (n == 0) { C[0] = C[1] = C[2] = C[3] = 0; bad = 0; nm = 0; drop = 0; }
            unsigned long long c_hi = ((unsigned long long)C[0] << 32) | C[1], c_lo = ((unsigned long long)C[2] << 32) | C[3];
            while (drop) {
                const int q = 63 - (__ffsll((long long)drop) - 1);       // last dropped position
                drop &= ~bit_at(q);
                // flag planes: bits after q move up by one
                const unsigned long long up = q ? ~from_pos(q) : 0ull;  // positions < q
                bad = (bad & up) | ((bad << 1) & ~up);
                nm = (nm & up) | ((nm << 1) & ~up);
                // code plane (128 bits, 2 per base)
                if (q < 32) {
                    const unsigned long long uph = q ? ~(~0ull >> (2 * q)) : 0ull;
                    c_hi = (c_hi & uph) | (((c_hi << 2) | (c_lo >> 62)) & ~uph);
                    c_lo <<= 2;
                } else {
                    const int q2 = q - 32;
                    const unsigned long long upl = q2 ? ~(~0ull >> (2 * q2)) : 0ull;
                    c_lo = (c_lo & upl) | ((c_lo << 2) & ~upl);
                }
            }
            C[0] = (uint32_t)(c_hi >> 32); C[1] = (uint32_t)c_hi; C[2] = (uint32_t)(c_lo >> 32); C[3] = (uint32_t)c_lo;
        }
        sm.keep[tid] = keep;
        int ktot;
        const int pos = block_exscan2(n, sm, ktot);
        sm.scan[tid] = pos;
        if (tid == 0) sm.ktot = ktot;
        // plain stores: every stream word whose first bit this thread covers
        const int u = PEND + pos;
        const int cw0 = u >> 4, csh = 2 * (u & 15), ncw = (csh + 2 * n + 31) >> 5;
        const int fw0 = u >> 5, fsh = u & 31, nfw = (fsh + n + 31) >> 5;
        uint32_t cwv[5], bwv[3], nwv[3];
        if (n > 0) {
            cwv[0] = C[0] >> csh;
            cwv[1] = __funnelshift_r(C[1], C[0], csh);
            cwv[2] = __funnelshift_r(C[2], C[1], csh);
            cwv[3] = __funnelshift_r(C[3], C[2], csh);
            cwv[4] = __funnelshift_r(0u, C[3], csh);
            const uint32_t bh = (uint32_t)(bad >> 32), bl = (uint32_t)bad, nh = (uint32_t)(nm >> 32), nlw = (uint32_t)nm;
            bwv[0] = bh >> fsh; bwv[1] = __funnelshift_r(bl, bh, fsh); bwv[2] = __funnelshift_r(0u, bl, fsh);
            nwv[0] = nh >> fsh; nwv[1] = __funnelshift_r(nlw, nh, fsh); nwv[2] = __funnelshift_r(0u, nlw, fsh);
            if (csh == 0) sm.cs[cw0] = cwv[0];
#pragma unroll
            for (int i = 1; i < 5; ++i) if (i < ncw) sm.cs[cw0 + i] = cwv[i];
            if (fsh == 0) { sm.bs[fw0] = bwv[0]; if (need_n) sm.ns[fw0] = nwv[0]; }
#pragma unroll
            for (int i = 1; i < 3; ++i) if (i < nfw) { sm.bs[fw0 + i] = bwv[i]; if (need_n) sm.ns[fw0 + i] = nwv[i]; }
        }
        __syncthreads();
        // partial first words are OR-ed in after the plain stores
        if (n > 0) {
            if (csh != 0 && cwv[0]) atomicOr(&sm.cs[cw0], cwv[0]);
            if (fsh != 0) {
                if (bwv[0]) atomicOr(&sm.bs[fw0], bwv[0]);
                if (need_n && nwv[0]) atomicOr(&sm.ns[fw0], nwv[0]);
            }
        }
        __syncthreads();

        // ---- 5. aggregate, look-back, inclusive prefix -----------------------------------------------------------
        int first_kept = ktot, last_kept = ktot;
        int closed_part = 0;
        if (m > 0) {
            first_kept = kept_before2(sm, (int)(rec_pos2(A, r_lo) - t0));
            last_kept = ktot - kept_before2(sm, (int)(rec_pos2(A, r_lo + m - 1) - t0));
            for (int e = tid; e < m - 1; e += NT) {
                int ka = kept_before2(sm, (int)(rec_pos2(A, r_lo + e) - t0));
                int kb = kept_before2(sm, (int)(rec_pos2(A, r_lo + e + 1) - t0));
                closed_part += tok_count32(kb - ka, P);
            }
        }
        int closed_tokens = 0;
        if (m > 1) (void)block_exscan2(closed_part, sm, closed_tokens);
        if (warp == 0) {
            const uint32_t tagA = (gen << 2) | ST_AGG, tagI = (gen << 2) | ST_INCL;
            const int k = P.k;
            Agg G;
            G.first = qr_of(first_kept, k); G.last = qr_of(last_kept, k); G.closed = closed_tokens; G.has_event = m > 0;
            const uint32_t tn = (uint32_t)min(k - 1, last_kept);
            uint64_t tl = 0;
            if (lane == 0) for (uint32_t i = 0; i < tn; ++i) tl = (tl << 4) | class_at(sm, PEND + ktot - (int)tn + (int)i);
            tl = __shfl_sync(0xffffffffu, tl, 0);
            G.tail = tl; G.tail_cnt = tn;
            Prefix X; X.T = 0; X.open.q = 0; X.open.r = 0; X.tail = 0; X.tail_cnt = 0;
            if (tile > 0) {
                if (lane == 0) {
                    st_vol128(&D.a0, make_uint4(tagA, (uint32_t)first_kept, (uint32_t)last_kept, (uint32_t)closed_tokens));
                    st_vol128(&D.a1, make_uint4(tagA, tn | ((uint32_t)(m > 0) << 8), (uint32_t)tl, (uint32_t)(tl >> 32)));
                }
                // warp-parallel look-back: lane l inspects tile base - l; one round trip per 32 tiles
                Agg acc; bool have = false, ok = true, done = false;
                for (int base = tile - 1; !done && ok; base -= 32) {
                    const int j = base - lane;
                    uint32_t st = ST_INCL;                   // tiles before 0 carry the empty inclusive prefix
                    Agg Aj; Prefix Xj;
                    Aj.first.q = Aj.last.q = Aj.closed = 0; Aj.first.r = Aj.last.r = 0; Aj.tail = 0; Aj.tail_cnt = 0; Aj.has_event = 0;
                    Xj.T = 0; Xj.open.q = 0; Xj.open.r = 0; Xj.tail = 0; Xj.tail_cnt = 0;
                    if (j >= 0) {
                        const TileDesc &Dj = A.descs[j];
                        int spins = 0;
                        for (;;) {
                            const uint4 w0 = ld_vol128(&Dj.i0), w1 = ld_vol128(&Dj.i1), w2 = ld_vol128(&Dj.i2);
                            const uint4 a0 = ld_vol128(&Dj.a0), a1 = ld_vol128(&Dj.a1);
                            if (w0.x == tagI && w1.x == tagI && w2.x == tagI) {
                                st = ST_INCL;
                                Xj.T = (int64_t)(((uint64_t)w0.w << 32) | w0.z);
                                Xj.tail_cnt = w0.y & 0xffu; Xj.open.r = (int32_t)(w0.y >> 8);
                                Xj.open.q = (int64_t)(((uint64_t)w1.w << 32) | w1.z);
                                Xj.tail = ((uint64_t)w2.w << 32) | w2.z;
                                break;
                            }
                            if (a0.x == tagA && a1.x == tagA) {
                                st = ST_AGG;
                                Aj.first = qr_of((int)a0.y, k); Aj.last = qr_of((int)a0.z, k); Aj.closed = (int64_t)a0.w;
                                Aj.tail_cnt = a1.y & 0xffu; Aj.has_event = a1.y >> 8;
                                Aj.tail = ((uint64_t)a1.w << 32) | a1.z;
                                break;
                            }
                            if (++spins > SPIN_LIMIT) { ok = false; break; }
                        }
                    }
                    ok = __all_sync(0xffffffffu, ok);
                    if (!ok) break;
                    const uint32_t ib = __ballot_sync(0xffffffffu, st == ST_INCL);
                    const int f = ib ? __ffs(ib) - 1 : 32;   // nearest tile with an inclusive prefix
                    if (lane >= f) {                         // identity element beyond the nearest inclusive prefix
                        Aj.first.q = Aj.last.q = Aj.closed = 0; Aj.first.r = Aj.last.r = 0; Aj.tail = 0; Aj.tail_cnt = 0; Aj.has_event = 0;
                    }
                    // ordered tree reduction: after the step of distance d lane l holds tiles [l, l + 2d) composed far -> near
#pragma unroll
                    for (int d = 1; d < 32; d <<= 1) {
                        Agg B;                               // what lane l + d holds: the farther (earlier) run
                        B.first.q = __shfl_down_sync(0xffffffffu, Aj.first.q, d);
                        B.last.q = __shfl_down_sync(0xffffffffu, Aj.last.q, d);
                        B.closed = __shfl_down_sync(0xffffffffu, Aj.closed, d);
                        B.tail = __shfl_down_sync(0xffffffffu, Aj.tail, d);
                        const uint32_t pk = (uint32_t)Aj.first.r | ((uint32_t)Aj.last.r << 4) | (Aj.tail_cnt << 8) | (Aj.has_event << 12);
                        const uint32_t pb = __shfl_down_sync(0xffffffffu, pk, d);
                        B.first.r = (int32_t)(pb & 15u); B.last.r = (int32_t)((pb >> 4) & 15u); B.tail_cnt = (pb >> 8) & 15u; B.has_event = pb >> 12;
                        if (lane + d < 32) Aj = agg_compose(B, Aj, P);
                    }
                    // lane 0 now holds this round's tiles; put it in front of what nearer rounds composed
                    if (f > 0) { acc = have ? agg_compose(Aj, acc, P) : Aj; have = true; }
                    if (f < 32) {
                        X.T = __shfl_sync(0xffffffffu, Xj.T, f); X.open.q = __shfl_sync(0xffffffffu, Xj.open.q, f);
                        X.open.r = __shfl_sync(0xffffffffu, Xj.open.r, f);
                        X.tail = __shfl_sync(0xffffffffu, Xj.tail, f); X.tail_cnt = __shfl_sync(0xffffffffu, Xj.tail_cnt, f);
                        done = true;
                    }
                }
                if (!ok && lane == 0) A.status[1] = 1u;
                if (have) X = prefix_apply(X, acc, P);       // valid in lane 0
            }
            if (lane == 0) {
                sm.pin = X;
                const Prefix Y = prefix_apply(X, G, P);
                st_vol128(&D.i0, make_uint4(tagI, Y.tail_cnt | ((uint32_t)Y.open.r << 8), (uint32_t)Y.T, (uint32_t)((uint64_t)Y.T >> 32)));
                st_vol128(&D.i1, make_uint4(tagI, 0u, (uint32_t)Y.open.q, (uint32_t)((uint64_t)Y.open.q >> 32)));
                st_vol128(&D.i2, make_uint4(tagI, 0u, (uint32_t)Y.tail, (uint32_t)(Y.tail >> 32)));
                // carried bases of the open record go in front of the stream
                const int pend = (P.mode == MODE_KMER) ? X.open.r : 0;
                uint32_t cw = 0, bw = 0, nw = 0;
                for (int i = 0; i < pend; ++i) {
                    const uint32_t c = (uint32_t)((X.tail >> (4 * (pend - 1 - i))) & 0xfu);
                    const int uu = PEND - pend + i;
                    if (c < CLS_N) cw |= c << (30 - 2 * uu);
                    else { bw |= 1u << (31 - uu); if (c == CLS_N) nw |= 1u << (31 - uu); }
                }
                sm.cs[0] = cw;
                if (bw) atomicOr(&sm.bs[0], bw);
                if (nw) atomicOr(&sm.ns[0], nw);
            }
        }
        __syncthreads();

        // ---- 6. emit ---------------------------------------------------------------------------------------------
        const Prefix X = sm.pin;
        const int pend = (P.mode == MODE_KMER) ? X.open.r : 0;
        {   // the record that was open at the tile's start: X.open.q of its windows were emitted by earlier tiles
            emit_segment2<IdT>(A, sm, PEND - pend, pend + first_kept, m > 0, A.out_bias + X.T + X.open.q, tid, NT);
        }
        if (m > 0) {
            int64_t base_T = A.out_bias + X.T + qr_tokens(qr_add(X.open, qr_of(first_kept, P.k), P.k), P);   // = out_offsets[r_lo]
            for (int c0 = 0; c0 < m; c0 += EV_CAP) {
                const int e = c0 + tid, cm = min(EV_CAP, m - c0);
                int ke = 0, ne = 0, te = 0;
                if (e < m) {
                    ke = kept_before2(sm, (int)(rec_pos2(A, r_lo + e) - t0));
                    int kn = (e + 1 < m) ? kept_before2(sm, (int)(rec_pos2(A, r_lo + e + 1) - t0)) : ktot;
                    ne = kn - ke;
                    te = (e + 1 < m) ? tok_count32(ne, P) : 0;
                }
                int chunk_total;
                int ex = block_exscan2(te, sm, chunk_total);
                if (e < m) {
                    A.out_off[r_lo + e] = base_T + ex;
                    sm.ev_k[tid] = ke; sm.ev_n[tid] = ne; sm.ev_out[tid] = base_T + ex;
                }
                __syncthreads();
                if (cm <= 8) {
                    for (int i = 0; i < cm; ++i)
                        if (r_lo + c0 + i < A.n_rec)
                            emit_segment2<IdT>(A, sm, PEND + sm.ev_k[i], sm.ev_n[i], c0 + i + 1 < m, sm.ev_out[i], tid, NT);
                } else {
                    for (int i = warp; i < cm; i += NW)
                        if (r_lo + c0 + i < A.n_rec)
                            emit_segment2<IdT>(A, sm, PEND + sm.ev_k[i], sm.ev_n[i], c0 + i + 1 < m, sm.ev_out[i], lane, 32);
                }
                base_T += chunk_total;
                __syncthreads();
            }
        }
    }
}

}  // namespace dtk
