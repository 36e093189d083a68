// encode_fasta.cuh -- the REGULAR-LAYOUT fast path of the strip encoder: classify + strip + {single-nt | k-mer} + CSR offsets
// for records whose layout is "optional '>' header line, then lines of one fixed width W, each ended by '\n'" (wrapped
// FASTA, one-line records, records of a single terminated line: BASELINE.json configs 1, 3, 5).
//
// For such a record the kept-base index of every byte is CLOSED FORM: with B = bytes of the header line and d = W + 1,
// byte x >= B is a base iff (x - B) mod d != W, and kidx(x) = ((x - B) div d) * W + min((x - B) mod d, W) bases precede it.
// So nothing has to be scanned across tiles: no chain, no look-back, no tickets, no block barrier.
//   fasta_parse_kernel    one thread per record reads its header line and its first sequence line (bounded), stores (B, W) and
//                         the record's token count; one thread per warp tile finds the record that holds the tile's first byte
//   offsets_scan_kernel   token counts -> out_offsets (chained scan over blocks of 2048 records)
//   encode_fasta_kernel   every WARP encodes whole 16 KiB tiles on its own: per record piece inside the tile it classifies 64
//                         bytes per lane exactly as encode_v5.cuh does, takes the keep mask from the closed form, compacts in
//                         registers, appends at the closed-form position into the warp's private kept-base stream in shared
//                         memory (interior words by shuffle + plain store, the two edge words by atomicOr), reads 64 bytes past
//                         the piece for the windows that straddle its end, and cuts the tokens whose first base lies in the piece.
// The closed form is an ASSUMPTION about the bytes, and every lane checks it on the bytes it holds: the SKIP bytes of the body
// must be exactly the predicted newlines, and no body line may start with '>' (which would be a second header line).  Any
// violation, a header or first line longer than the parse bound, or more than 16 records in one tile, sets *irregular; the
// chained-scan encoder of encode_v5.cuh is launched behind this kernel in every call and returns at once unless the flag
// is set, in which case it encodes the whole input again (the result is then its result).  The LUT stays the specification:
// a table with other SKIP bytes, or one that does not skip '\n', simply fails the check wherever such bytes occur.
#pragma once
#include "encode_v5.cuh"
#include "encode_v7.cuh"

namespace dtk {
namespace fa {

using namespace dtk::v5;

// (compile-time knobs for tuning sweeps -- DTK_NVCC_FLAGS="-DFW_WARPS_N=4 -DFW_CHUNKS_N=6 -DFW_MINB=7" -- the defaults are the
// measured optimum)
#ifndef FW_CHUNKS_N
#define FW_CHUNKS_N 8
#endif
#ifndef FW_WARPS_N
#define FW_WARPS_N 8
#endif
#ifndef FW_MINB
#define FW_MINB 3
#endif
constexpr int FW_CHUNKS = FW_CHUNKS_N;               // 2 KiB chunks per warp tile
constexpr int FW_TILE = FW_CHUNKS * WB;             // bytes per warp tile (16 KiB)
constexpr int FW_HALO = 64;                         // bytes read past a piece that ends at the tile's end
constexpr int FW_BASES = FW_TILE + FW_HALO;
constexpr int FW_CW = FW_BASES / 16 + 8;            // code words of a warp's stream (+ over-read slack)
constexpr int FW_FW = FW_BASES / 32 + 10;
constexpr int FW_WORDS = FW_CW + FW_FW;
constexpr int FW_WARPS = FW_WARPS_N;                 // warps per CTA
constexpr int FW_MAXSEG = 2 * FW_CHUNKS;            // records per warp tile the fast path accepts
constexpr int FW_HDR_BOUND = 4096;                  // bytes the parse reads looking for the end of a header line
constexpr int FW_LINE_BOUND = 512;                  //   ... and for the end of the first sequence line
static_assert(FW_WORDS % 4 == 0, "per-warp streams stay 16-byte aligned");

struct FastaArgs {
    EncArgs e;
    int32_t *par;                // [n_rec][4]: B (bytes of the header line, 0 if none), W (line width; >= 1), Z (1: the record's
                                 //             last byte is the line end of its last line), dmul (floor(2^32 / (W + 1)) + 1, or 0
                                 //             if W + 1 > 65536)
    int32_t *rec_tok;            // [n_rec] tokens of every record
    int32_t *wt_first;           // [n_wtiles] record that holds the tile's first byte (first record starting behind it if none)
    uint32_t *irregular;         // set when the input does not have the regular layout
    int32_t n_wtiles;
    // seq_len > 0: the tokens go straight into the padded batch (e.ids = batch_ids[n_rec][seq_len] int32, e.ids_cap = n_rec * seq_len):
    // token j < seq_len of record r at column j + (pad_side == 0 ? seq_len - min(tokens, seq_len) : 0) -- pad_kernel.cuh's rule; the
    // pad columns and the mask are pad_fill_kernel's
    int32_t seq_len, pad_side;
};

struct SmemFa {
    uint32_t strm[FW_WARPS][FW_WORDS];
    uint4 stage[FW_WARPS][4 * 32];      // the chunk a warp works on next, copied asynchronously: 16-byte unit j of lane l at [j * 32 + l]
    uint8_t lut[256];
};

// this lane's 64 bytes of the chunk at tile offset c (tile base tb) -> the warp's staging buffer; bytes from tile offset lim on
// read as zero.  One cp.async group per chunk.
__device__ __forceinline__ void stage_chunk(uint4 *stg, const uint8_t *tb, int c, int lim, int lane) {
    const int q = c + lane * LB;
    const uint32_t dst = (uint32_t)__cvta_generic_to_shared(stg + lane);
    const uint8_t *src = tb + q;
    if (c + WB <= lim) {                                         // the whole chunk lies inside the input (warp-uniform)
#pragma unroll
        for (int j = 0; j < 4; ++j)
            asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst + j * 512), "l"(src + 16 * j) : "memory");
    } else {
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const int sz = q + 16 * j < lim ? 16 : 0;
            asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(dst + j * 512), "l"(src + 16 * j), "r"(sz) : "memory");
        }
    }
    asm volatile("cp.async.commit_group;" ::: "memory");
}

// bases among the first y body bytes of a record with line width W
__device__ __forceinline__ int64_t kept_before(int64_t y, int W) {
    if (y <= 0) return 0;
    const int64_t d = (int64_t)W + 1, line = y / d, col = y - line * d;
    return line * W + (col < W ? col : W);
}

// position of the first '\n' among the bytes al[from, to), or `to` if there is none; al is 16-byte aligned and is read 16 bytes
// at a time (up to 15 bytes past `to`, like every other kernel here).  A byte equals '\n' iff its XOR with 0x0A is zero; the
// lowest flag of the classic zero-byte test is exact (a false flag can only sit above a true one).
__device__ __forceinline__ int64_t find_nl(const uint8_t *al, int64_t from, int64_t to) {
    // 64 bytes per step: the four loads of a step are independent, so a long first line costs a quarter of the round trips
    for (int64_t p = from & ~(int64_t)15; p < to; p += 64) {
        uint4 v[4];
#pragma unroll
        for (int i = 0; i < 4; ++i) v[i] = p + 16 * i < to ? __ldg(reinterpret_cast<const uint4 *>(al + p + 16 * i)) : make_uint4(0, 0, 0, 0);
        const uint32_t *w = reinterpret_cast<const uint32_t *>(v);
#pragma unroll
        for (int j = 0; j < 16; ++j) {
            const uint32_t y = w[j] ^ 0x0A0A0A0Au;
            uint32_t z = (y - 0x01010101u) & ~y & 0x80808080u;
            const int64_t wp = p + 4 * j;
            if (wp < from) z = from - wp >= 4 ? 0u : z & (0xffffffffu << (8 * (int)(from - wp)));
            if (z) { const int64_t pos = wp + ((__ffs((int)z) - 1) >> 3); return pos < to ? pos : to; }
        }
    }
    return to;
}

__global__ void __launch_bounds__(256) fasta_parse_kernel(const __grid_constant__ FastaArgs F) {
    const EncArgs &A = F.e;
    const EncParams &P = A.prm;
    // threads [0, n_wtiles) search for the first record of a tile, threads [n_wtiles, n_wtiles + n_rec) parse a record each: two
    // short chains of dependent loads side by side instead of one long one per thread
    const int64_t t0 = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    if (t0 < F.n_wtiles) {
        const int64_t t = t0;
        // last record whose start is at or before the tile's first byte (0 if the tile starts in front of every record)
        const int64_t pos = t * FW_TILE;
        // number of offsets <= pos, by a 16-way search: the 16 probes of a step are independent loads, so the chain of
        // dependent memory round trips is log16 instead of log2 of the record count
        int64_t lo = 0, hi = A.n_rec + 1;                       // every m < lo has offset <= pos, no m >= hi has
        while (lo < hi) {
            const int64_t step = (hi - lo + 15) >> 4;
            bool le[16];
#pragma unroll
            for (int i = 0; i < 16; ++i) { const int64_t m = lo + i * step; le[i] = m < hi && rec_pos(A, m) <= pos; }
            int c = 0;
#pragma unroll
            for (int i = 0; i < 16; ++i) c += le[i] ? 1 : 0;    // the probes that hold form a prefix (offsets ascend)
            if (c == 0) { hi = lo; break; }
            const int64_t nhi = lo + c * step;                  // the first probe that fails, if one was made
            lo = lo + (c - 1) * step + 1;
            if (c < 16 && nhi < hi) hi = nhi;
        }
        F.wt_first[t] = (int32_t)(lo > 0 ? lo - 1 : 0);
        return;
    }
    const int64_t t = t0 - F.n_wtiles;
    if (t >= A.n_rec) return;
    const int64_t a = rec_pos(A, t), e = rec_pos(A, t + 1), L = e - a;
    const uint8_t *b = A.bytes_al + a;
    bool bad = L >= (1ll << 31);
    const uint32_t last_byte = L > 0 ? (uint32_t)__ldg(b + L - 1) : 0u;     // asked for early: a cache line of its own
    const bool nl_skipped = __ldg(F.e.lut + (uint8_t)'\n') == CLS_SKIP;
    int64_t B = 0;
    if (P.strip_headers && L > 0 && b[0] == '>') {
        const int64_t lim = L < FW_HDR_BOUND ? L : FW_HDR_BOUND;
        const int64_t i = find_nl(A.bytes_al, a + 1, a + lim) - a;
        if (i < lim) B = i + 1;                                 // through the '\n'
        else if (lim == L) B = L;                               // a header with no line end runs to the record's end (Q4)
        else bad = true;
    }
    // a record's last line is usually shorter than the others: its line end, the record's last byte, is set apart
    int64_t Z = 0;
    if (L - B > 0 && last_byte == '\n' && nl_skipped) Z = 1;
    const int64_t body = L - B - Z;
    int64_t W = body;                                           // one line without a line end
    if (body > 0) {
        const int64_t lim = body < FW_LINE_BOUND ? body : FW_LINE_BOUND;
        const int64_t i = find_nl(A.bytes_al, a + B, a + B + lim) - (a + B);
        if (i < lim) W = i;
        // (else: a long single line; the encode kernel checks that it holds no line end)
    }
    if (W < 1) { W = 1; if (body > 0) bad = true; }             // a body that starts with an empty line is not regular
    if (bad) { *F.irregular = 1u; B = 0; W = 1; Z = 0; }
    const int64_t Wc = W > 0x7fffffff ? 0x7fffffff : W, dd = Wc + 1;
    const uint32_t dmul = dd <= 65536 ? (uint32_t)(0x100000000ull / (unsigned long long)dd) + 1u : 0u;    // see div_d below
    reinterpret_cast<int4 *>(F.par)[t] = make_int4((int32_t)B, (int32_t)Wc, (int32_t)Z, (int32_t)dmul);
    const int64_t n = bad ? 0 : kept_before(body, (int)W);
    int64_t tok = n;
    if (P.mode == MODE_KMER) { const int64_t q = n / P.k; tok = q + tail_tokens((int)(n - q * P.k), P); }
    F.rec_tok[t] = (int32_t)(tok > 0x7fffffff ? 0x7fffffff : tok);
}

// out_offsets = exclusive scan of per-record token counts; chained over blocks of 2048 records (chain words: a0 of the tile
// descriptors { tag, 0, sum lo, sum hi }, generation-tagged like everything else in that array)
constexpr int OS_NT = 256, OS_PER = 8, OS_BLK = OS_NT * OS_PER;
__global__ void __launch_bounds__(OS_NT) offsets_scan_kernel(const int32_t *tok, int64_t n_rec, int64_t *out_off, int64_t out_bias,
                                                            TileDesc *chain, uint32_t gen, uint32_t *status) {
    __shared__ long long wsum[OS_NT / 32];
    __shared__ long long s_base;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    asm volatile("griddepcontrol.wait;" ::: "memory");
    const int b = (int)blockIdx.x;
    const int64_t r0 = (int64_t)b * OS_BLK + (int64_t)tid * OS_PER;
    long long v[OS_PER], run = 0;
#pragma unroll
    for (int i = 0; i < OS_PER; ++i) { v[i] = r0 + i < n_rec ? tok[r0 + i] : 0; run += v[i]; }
    long long inc = run;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) { const long long t = __shfl_up_sync(0xffffffffu, inc, d); if (lane >= d) inc += t; }
    if (lane == 31) wsum[warp] = inc;
    __syncthreads();
    long long woff = 0, tot = 0;
#pragma unroll
    for (int w = 0; w < OS_NT / 32; ++w) { const long long t = wsum[w]; if (w < warp) woff += t; tot += t; }
    const uint32_t tagA = (gen << 2) | ST_AGG, tagI = (gen << 2) | ST_INCL;
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
                    if (++spins > SPIN_LIMIT) { status[1] = 1u; break; }
                    __nanosleep(20);
                }
                base += (long long)(((unsigned long long)w.w << 32) | w.z);
                if (w.x == tagI) break;
            }
        }
        const long long incl = base + tot;
        st_vol128(&chain[b].a0, make_uint4(tagI, 0u, (uint32_t)incl, (uint32_t)((unsigned long long)incl >> 32)));
        s_base = base;
        if ((int64_t)(b + 1) * OS_BLK >= n_rec) out_off[n_rec] = out_bias + incl;
    }
    __syncthreads();
    long long ex = s_base + woff + inc - run + out_bias;
#pragma unroll
    for (int i = 0; i < OS_PER; ++i) { if (r0 + i < n_rec) out_off[r0 + i] = ex; ex += v[i]; }
}

// ---- the columns of the padded batch that hold no token, and the whole mask, from the token counts alone (fused path: the
// encoder behind writes the tokens into their columns itself).  One CTA per row, four columns per thread and step. ----
struct PadFillArgs {
    const int64_t *out_off; int64_t n_rows;
    int32_t *batch_ids; uint8_t *mask;          // mask may be null
    int32_t seq_len, pad_side, pad_id;
};
__global__ void __launch_bounds__(256) pad_fill_kernel(const __grid_constant__ PadFillArgs A) {
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    asm volatile("griddepcontrol.wait;" ::: "memory");           // out_offsets come from the scan in front
    const int L = A.seq_len;
    const bool vec = (L & 3) == 0 && (reinterpret_cast<uintptr_t>(A.batch_ids) & 15) == 0 &&
                     (A.mask == nullptr || (reinterpret_cast<uintptr_t>(A.mask) & 3) == 0);
    for (int64_t r = blockIdx.x; r < A.n_rows; r += gridDim.x) {
        const int64_t tok = A.out_off[r + 1] - A.out_off[r];
        const int m = (int)(tok < L ? tok : L);
        const int col0 = A.pad_side == 0 ? L - m : 0;            // the kept tokens sit in columns [col0, col0 + m)
        int32_t *row = A.batch_ids + r * L;
        uint8_t *mrow = A.mask ? A.mask + r * L : nullptr;
        if (vec) {
            for (int c = threadIdx.x * 4; c < L; c += blockDim.x * 4) {
                uint32_t mk = 0;
                int n_in = 0;
#pragma unroll
                for (int j = 0; j < 4; ++j) { const bool in = c + j >= col0 && c + j < col0 + m; mk |= (uint32_t)in << (8 * j); n_in += in; }
                if (n_in == 0) *reinterpret_cast<int4 *>(row + c) = make_int4(A.pad_id, A.pad_id, A.pad_id, A.pad_id);
                else if (n_in < 4) {
#pragma unroll
                    for (int j = 0; j < 4; ++j) if (!((mk >> (8 * j)) & 1u)) row[c + j] = A.pad_id;
                }
                if (mrow) *reinterpret_cast<uint32_t *>(mrow + c) = mk;
            }
        } else {
            for (int c = threadIdx.x; c < L; c += blockDim.x) {
                const bool in = c >= col0 && c < col0 + m;
                if (!in) row[c] = A.pad_id;
                if (mrow) mrow[c] = in ? 1 : 0;
            }
        }
    }
}

// ---- emission from a warp's private stream (code words cw, flag words fw; base u at bits 31-2(u&15).. of cw[u>>4]) ----
// FLAGS = false: the caller knows that no base of the piece is flagged (the flag words are not read)
template <typename IdT, int K, bool SINGLE, bool REMAP, bool FLAGS = true>
__device__ __forceinline__ void emit_group_w(const EncArgs &A, const uint32_t *cw, const uint32_t *fw, int o, IdT *dst, bool affine) {
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
    if (FLAGS) {
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
        else id[t] = (REMAP && P.remap4) ? __ldg(P.remap4 + c[t]) : P.base_id + (int32_t)c[t];
    }
    if (FLAGS && anybad) {
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

__device__ __forceinline__ uint32_t w_code(const uint32_t *cw, int u, int k) {       // k <= 15 digits starting at base u
    const int b = 2 * u, w = b >> 5, s = b & 31;
    return __funnelshift_l(cw[w + 1], cw[w], s) >> (32 - 2 * k);
}
__device__ __forceinline__ uint32_t w_flags(const uint32_t *fw, int u, int k) {
    const int w = u >> 5, s = u & 31;
    return __funnelshift_l(fw[w + 1], fw[w], s) >> (32 - k);
}
__device__ __forceinline__ uint32_t w_class(const uint32_t *cw, const uint32_t *fw, int u) {
    const uint32_t c = w_code(cw, u, 1);
    return w_flags(fw, u, 1) ? (c == 2u ? CLS_N : CLS_UNK) : c;
}
// id of window j (its k bases start at stream position u)
__device__ __forceinline__ int32_t w_window_id(const EncParams &P, const uint32_t *cw, const uint32_t *fw, int u) {
    if (P.mode != MODE_KMER) { const uint32_t c = w_class(cw, fw, u); return c <= CLS_N ? P.nt_ids[c] : P.unk_id; }
    const uint32_t fl = w_flags(fw, u, P.k), cd = w_code(cw, u, P.k);
    return P.remap4 ? kmer_table_id_cold(P, cd, fl, P.k) : (fl ? P.unk_id : (int32_t)(P.base_id + cd));
}

template <typename IdT, int KK>
__device__ __forceinline__ void emit_group_sel(const EncArgs &A, const uint32_t *cw, const uint32_t *fw, int u, IdT *dst, bool affine, int kk,
                                               bool flags) {
    if constexpr (KK == 0) emit_group_w<IdT, 1, true, false>(A, cw, fw, u, dst, affine);
    else if constexpr (KK > 0) {
        if (flags) emit_group_w<IdT, KK, false, false, true>(A, cw, fw, u, dst, false);
        else emit_group_w<IdT, KK, false, false, false>(A, cw, fw, u, dst, false);
    }
    else switch (kk) {
        case 0: emit_group_w<IdT, 1, true, false>(A, cw, fw, u, dst, affine); break;
        case 1: emit_group_w<IdT, 1, false, true>(A, cw, fw, u, dst, false); break;
        case 2: emit_group_w<IdT, 2, false, true>(A, cw, fw, u, dst, false); break;
        case 3: emit_group_w<IdT, 3, false, true>(A, cw, fw, u, dst, false); break;
        case 4: emit_group_w<IdT, 4, false, true>(A, cw, fw, u, dst, false); break;
        case 5: emit_group_w<IdT, 5, false, true>(A, cw, fw, u, dst, false); break;
        case 6: emit_group_w<IdT, 6, false, true>(A, cw, fw, u, dst, false); break;
        default: emit_group_w<IdT, 8, false, true>(A, cw, fw, u, dst, false); break;
    }
}

// y / d for any 32-bit y by one multiply-high and a correction: with dmul = floor(2^32 / d) + 1 the estimate is the quotient or
// one more (y dmul / 2^32 = y / d + y e / (d 2^32), e = dmul d - 2^32 <= d).  dmul == 0 (d > 65536): the division itself.
__device__ __forceinline__ uint32_t div_d(uint32_t y, uint32_t d, uint32_t dmul) {
    if (dmul == 0u) return y / d;
    uint32_t q = __umulhi(y, dmul);
    if (q * d > y) --q;
    return q;
}

__device__ __forceinline__ int clamp64(int64_t v) { return v < 0 ? 0 : (v > 64 ? 64 : (int)v); }

// ======================================================================================================
// KK: the emission variant compiled in -- 0 single-nt, 1..6 / 8 that k, -1 every variant behind a run-time switch
// FUSED: the tokens go into the padded batch (FastaArgs::seq_len > 0; IdT = int32_t)
template <typename IdT, int KK, bool FUSED = false>
__global__ void __launch_bounds__(FW_WARPS * 32, FW_MINB) encode_fasta_kernel(const __grid_constant__ FastaArgs F) {
    extern __shared__ __align__(16) uint8_t smem_raw[];
    SmemFa &sm = *reinterpret_cast<SmemFa *>(smem_raw);
    constexpr uint32_t FULL = 0xffffffffu;
    constexpr int R = 16 / (int)sizeof(IdT);
    const EncArgs &A = F.e;
    const EncParams &P = A.prm;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int k = KK > 0 ? KK : (P.mode == MODE_KMER ? P.k : 1);       // a compile-time constant in the per-k variants
    const int kk = P.mode == MODE_KMER ? k : 0;
    const bool affine = P.nt_ids[1] == P.nt_ids[0] + 1 && P.nt_ids[2] == P.nt_ids[0] + 2 && P.nt_ids[3] == P.nt_ids[0] + 3;
    const bool vec_ok = (reinterpret_cast<uintptr_t>(A.ids) & 15) == 0 &&
                        (P.mode != MODE_KMER || (k >= 1 && k <= 6) || k == 8);
    for (int i = tid; i < 256; i += FW_WARPS * 32) sm.lut[i] = A.lut[i];
    __syncthreads();
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    {   // the warp's first tile on its way to L2 while the parse and scan kernels in front still run (HBM idles meanwhile)
        const int64_t p0 = ((int64_t)blockIdx.x * FW_WARPS + warp) * FW_TILE;
        int64_t sz = A.p_end - p0; if (sz > FW_TILE) sz = FW_TILE; sz &= ~(int64_t)15;
        if (lane == 0 && sz > 0) asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(A.bytes_al + p0), "r"((uint32_t)sz) : "memory");
    }
    asm volatile("griddepcontrol.wait;" ::: "memory");           // par, wt_first, out_offsets come from the kernels in front
    uint32_t *const cw = sm.strm[warp], *const fw = cw + FW_CW;
    IdT *const ids = reinterpret_cast<IdT *>(A.ids);
    bool irregular = false;
    const bool nl_skips = sm.lut[(uint8_t)'\n'] == CLS_SKIP;

    // Tiles are handed out through a counter (F.irregular + 2, zeroed with the flag): the first one of a warp is its own index,
    // every later one is taken when the warp starts the tile before it, so that no SM is left idle while others still have
    // several tiles of uneven cost in front of them.  (No L2 prefetch: with the next chunk always in flight it bought no time
    // and cost a fifth more DRAM reads.)
    const int64_t n_warps = (int64_t)gridDim.x * FW_WARPS;
    unsigned long long *const tile_ctr = reinterpret_cast<unsigned long long *>(F.irregular + 2);
    int64_t tile = (int64_t)blockIdx.x * FW_WARPS + warp;
#pragma unroll 1
    while (tile < F.n_wtiles) {
        // somebody has found the layout irregular: the chained-scan encoder will redo everything, so stop here
        if (__ldcg(F.irregular) != 0u) break;
        int64_t next_tile = 0;
        if (lane == 0) next_tile = n_warps + (int64_t)atomicAdd(tile_ctr, 1ull);
        next_tile = __shfl_sync(FULL, next_tile, 0);
        const int64_t ts = tile * FW_TILE, te = ts + FW_TILE < A.p_end ? ts + FW_TILE : A.p_end;
        int nseg = 0;
#pragma unroll 1
        for (int64_t r = F.wt_first[tile]; r < A.n_rec; ++r) {
            const int64_t rs = rec_pos(A, r);
            if (rs >= te) break;
            const int64_t re = rec_pos(A, r + 1);
            const int64_t sa = rs > ts ? rs : ts, sb = re < te ? re : te;       // the record's piece inside this tile
            if (sb <= sa) continue;
            if (++nseg > FW_MAXSEG) { irregular = true; break; }
            const int4 par = __ldg(reinterpret_cast<const int4 *>(F.par) + r);
            const int B = par.x, W = par.y, Z = par.z;
            const uint32_t d = (uint32_t)W + 1u;
            // c / d in one multiply for the columns c < d + FW_TILE + FW_HALO met below: exact while c * (dmul * d - 2^32) < 2^32
            // (every d up to 2^14) or c < 2 d - 1 (the larger d)
            const uint32_t dmul = (uint32_t)par.w;
            const int64_t bend = re - Z;                                         // end of the body (the record's final line end set apart)
            const int64_t sbb = sb < bend ? sb : bend;
            // everything below is 32 bits wide and relative to the tile's first byte
            const int sa_rel = (int)(sa - ts);
            int64_t he = sb;                                                     // bytes behind a piece that ends at the tile's end:
            if (sb == te && re > sb) { he = sb + FW_HALO; if (he > A.p_end) he = A.p_end; }   //   the windows that start in the piece run into them
            if (he > bend) he = bend;
            int he_rel = (int)(he - ts);
            const int64_t yb = ts - rs - B;                                      // body index of the tile's first byte (may be negative)
            // body index, line and column of the piece's first body byte; bases of the record in front of / through the piece
            const uint32_t y_p = (uint32_t)(sa - rs > B ? sa - rs - B : 0);
            const uint32_t line_p = div_d(y_p, d, dmul), col_p = y_p - line_p * d;
            // (a record is shorter than 2^31 bytes -- the parse kernel flags anything longer -- so base counts fit 32 bits)
            const uint32_t K0 = line_p * (uint32_t)W + col_p;
            const uint32_t y_e = (uint32_t)(sbb - rs > B ? sbb - rs - B : 0);
            const uint32_t line_e = div_d(y_e, d, dmul), col_e = y_e - line_e * d;
            const int nK = (int)(line_e * (uint32_t)W + col_e - K0);             // bases of the piece
            // windows of the record: only matters when the record ends near the piece
            constexpr uint32_t FAR = 0xffffffffu;
            uint32_t nwin = FAR, n_r = FAR;
            if (re - sb < 2 * FW_HALO) {
                const uint32_t y_r = (uint32_t)(bend - rs > B ? bend - rs - B : 0);
                const uint32_t line_r = div_d(y_r, d, dmul), col_r = y_r - line_r * d;
                n_r = line_r * (uint32_t)W + col_r;
                nwin = n_r / (uint32_t)k;
            }
            const int64_t T_r = __ldcg(A.out_off + r);
            // destination index of the record's token 0, and the number of its tokens that have a place at all
            int64_t g_base = T_r;
            uint32_t jcap = 0xffffffffu;
            if (FUSED) {
                const int64_t Ttok = __ldcg(A.out_off + r + 1) - T_r, L = F.seq_len;
                g_base = r * L + (F.pad_side == 0 ? L - (Ttok < L ? Ttok : L) : 0);
                jcap = (uint32_t)L;
            }
            // the warp's stream starts empty (edge words are OR-ed in)
            for (int i = lane; i < FW_WORDS / 4; i += 32) reinterpret_cast<uint4 *>(cw)[i] = make_uint4(0, 0, 0, 0);
            __syncwarp();
            const uint8_t *const tb = A.bytes_al + ts;
            const int end_rel = A.p_end - ts > (1 << 20) ? (1 << 20) : (int)(A.p_end - ts);
            const int lim_rel = end_rel;                                         // bytes from here on read as zero
            uint4 *const stg = sm.stage[warp];
            bool has_flags = false;
            // ---- the bytes behind a piece that ends at the tile's end.  Only the k - 1 <= 14 bases that the piece's last windows
            // run into are needed, and the warp that owns the next tile is the one that checks them.  Wrapped lines of ACGT: 16
            // bytes, classified by every lane alike, at most one predicted line end dropped, appended by lane 0 at stream
            // position nK.  Anything else (an N among them, a header, short lines) goes through the chunk loop below. ----
            if (he - sb >= 16 && d >= 65u && P.fast_lut && nl_skips && yb + (sb - ts) >= 0) {
                const int sb_rel = (int)(sb - ts);
                const uint4 hv = __ldg(reinterpret_cast<const uint4 *>(tb + sb_rel));
                const uint32_t c = col_p + ((uint32_t)(yb + sb_rel) - y_p);
                const uint32_t q = dmul ? __umulhi(c, dmul) : (uint32_t)(c >= d);
                const uint32_t tn = (uint32_t)W - (c - q * d);                    // offset of the predicted line end (>= 16: none here)
                const uint32_t xw[4] = {hv.x, hv.y, hv.z, hv.w};
                uint32_t cb[4], inval = 0u;
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    const uint32_t x = xw[j];
                    cb[j] = (x & 0x06060606u) * 0x00820820u;
                    const uint32_t m = (x >> 2) & ~(x >> 1) & 0x01010101u;
                    uint32_t dj = (x & 0xD9D9D9D9u) ^ (m * 0x0fu + 0x41414141u);
                    if ((tn >> 2) == (uint32_t)j) dj &= ~(0xffu << (8 * (tn & 3u)));
                    inval |= dj;
                }
                if (inval == 0u) {
                    const uint32_t lo2 = __byte_perm(cb[0], cb[1], 0x0073), hi2 = __byte_perm(cb[2], cb[3], 0x0073);
                    const uint32_t y = __brev(__byte_perm(lo2, hi2, 0x5410));
                    uint32_t C = ((y & 0x55555555u) << 1) | (((y >> 1) ^ y) & 0x55555555u);
                    if (tn < 16u) { const uint32_t T = ~(0xffffffffu >> (2 * tn)); C = (C & T) | ((C << 2) & ~T); }
                    if (lane == 0) {
                        const int sh = 2 * (nK & 15);
                        atomicOr(&cw[nK >> 4], C >> sh);
                        if (sh) atomicOr(&cw[(nK >> 4) + 1], C << (32 - sh));
                    }
                    he_rel = sb_rel;                                             // the chunk loop stops at the tile's end
                }
            }
            if ((sa_rel & ~(WB - 1)) < he_rel) stage_chunk(stg, tb, sa_rel & ~(WB - 1), lim_rel, lane);
            // chunks [lean_lo, lean_hi) of the piece may take the lean road below: whole chunks of body bytes inside the input
            // (lean_hi: the last one may be the 64-byte multiple read past the tile's end)
            int lean_lo = 1 << 30, lean_hi = 0;
            if (d >= 65u && P.fast_lut && nl_skips) {
                lean_lo = (sa_rel + WB - 1) & ~(WB - 1);
                if (yb + lean_lo < 0) lean_lo = (int)((-yb + WB - 1) & ~(int64_t)(WB - 1));
                const int full_end = min(he_rel, end_rel) & ~(WB - 1);            // end of the last whole chunk
                lean_hi = full_end;
                const int rest = he_rel - full_end;
                if (rest > 0 && (rest & 63) == 0 && he_rel <= end_rel) lean_hi = full_end + WB;
            }
#pragma unroll 1
            for (int c_rel = sa_rel & ~(WB - 1); c_rel < he_rel; c_rel += WB) {
                const int q_rel = c_rel + lane * LB;                             // tile offset of this lane's first byte
                // this chunk's bytes arrive from the staging buffer; the next chunk's copy starts before the work on this one
                asm volatile("cp.async.wait_group 0;" ::: "memory");
                // ---- interior chunk of wrapped lines (the bulk of a FASTA record): all 2 KiB are body bytes of the piece, lines
                // are longer than a lane, so each lane holds 64 body bytes and at most one predicted line end.  Streamlined:
                // no per-byte flags, no masks; falls through to the general code below if any lane fails the layout check ----
                // The 64 bytes read past the tile's end take the same road with one active lane (nact = active lanes).
                const int left = he_rel - c_rel;
                const bool lean = c_rel >= lean_lo && c_rel < lean_hi;
                const int nact = left >= WB ? 32 : left >> 6;
                const bool on = lane < nact;
                uint32_t tn = 64u;                                               // lane index of the predicted line end (>= 64: none)
                int u = 0;
                bool probe_ok = true;
                if (lean) {
                    const uint32_t c = col_p + ((uint32_t)(yb + q_rel) - y_p);   // column counted from the piece's first line
                    const uint32_t q = dmul ? __umulhi(c, dmul) : (uint32_t)(c >= d);
                    const uint32_t col = c - q * d;
                    if (on) tn = (uint32_t)W - col;
                    u = (int)(q * (uint32_t)W + col) - (int)col_p;
                    if (tn < 64u) {
                        // the byte where the closed form puts the line end must be '\n'; in the staging buffer it becomes an 'A',
                        // so that the classification below has one question to ask of all 64 bytes, and its code is deleted later
                        uint8_t *pb = reinterpret_cast<uint8_t *>(stg + (tn >> 4) * 32 + lane) + (tn & 15u);
                        probe_ok = *pb == '\n';
                        *pb = 'A';
                    }
                }
                uint4 v[4];
#pragma unroll
                for (int j = 0; j < 4; ++j) v[j] = stg[j * 32 + lane];
                if (c_rel + WB < he_rel) stage_chunk(stg, tb, c_rel + WB, lim_rel, lane);
                if (lean) {
                    if (!on) { v[0] = v[1] = v[2] = v[3] = make_uint4(0x41414141u, 0x41414141u, 0x41414141u, 0x41414141u); }
                    uint32_t C[4], dd[16];
                    {
                        const uint32_t *xw = reinterpret_cast<const uint32_t *>(v);
                        uint32_t cb[16];
#pragma unroll
                        for (int j = 0; j < 16; ++j) {
                            const uint32_t x = xw[j];
                            cb[j] = (x & 0x06060606u) * 0x00820820u;
                            const uint32_t m = (x >> 2) & ~(x >> 1) & 0x01010101u;       // (as IMAD.HI on the FMA pipe: 1 % slower)
                            dd[j] = (x & 0xD9D9D9D9u) ^ (m * 0x0fu + 0x41414141u);
                        }
#pragma unroll
                        for (int h = 0; h < 4; ++h) {
                            const uint32_t lo2 = __byte_perm(cb[4 * h], cb[4 * h + 1], 0x0073);
                            const uint32_t hi2 = __byte_perm(cb[4 * h + 2], cb[4 * h + 3], 0x0073);
                            const uint32_t y = __brev(__byte_perm(lo2, hi2, 0x5410));
                            C[h] = ((y & 0x55555555u) << 1) | (((y >> 1) ^ y) & 0x55555555u);
                        }
                    }
                    uint32_t any = 0u;
#pragma unroll
                    for (int j = 0; j < 16; ++j) any |= dd[j];
                    const bool ok = probe_ok && any == 0u;
                    if (__all_sync(FULL, ok)) {
                        int n = 64;
                        if (tn < 64u) {                                          // the line end leaves the code plane
                            n = 63;
                            const int q2 = 2 * (int)tn;
#pragma unroll
                            for (int j = 0; j < 4; ++j) {
                                const uint32_t nx = j < 3 ? C[j + 1] : 0u;
                                const uint32_t S = __funnelshift_l(nx, C[j], 2);
                                const uint32_t T = __funnelshift_rc(0xffffffffu, 0u, max(q2 - 32 * j, 0));
                                C[j] = (C[j] & ~T) | (S & T);
                            }
                        }
                        // every base is one of ACGT: the flag words stay zero; code words as in the general append below
                        const int cw0 = u >> 4, csh = 2 * (u & 15), cend = csh + 2 * n;
                        const uint32_t w0 = C[0] >> csh, w1 = __funnelshift_r(C[1], C[0], csh), w2 = __funnelshift_r(C[2], C[1], csh),
                                       w3 = __funnelshift_r(C[3], C[2], csh), w4 = __funnelshift_r(0u, C[3], csh);
                        const int li = cend >> 5;
                        uint32_t part = li == 2 ? w2 : (li == 3 ? w3 : w4);
                        if ((cend & 31) == 0) part = 0u;
                        const uint32_t prev = __shfl_up_sync(FULL, part, 1);
                        if (on) {
                            if (lane == 0) { if (w0) atomicOr(&cw[cw0], w0); } else cw[cw0] = w0 | prev;
                            cw[cw0 + 1] = w1;
                            if (cend >= 96) cw[cw0 + 2] = w2;
                            if (cend >= 128) cw[cw0 + 3] = w3;
                            if (lane == nact - 1 && part) atomicOr(&cw[cw0 + li], part);
                        }
                        continue;
                    }
                    // some byte is not one of ACGT (an N, say): the general code takes the chunk, on the bytes as they are in memory
                    const uint4 *src = reinterpret_cast<const uint4 *>(tb + q_rel);
#pragma unroll
                    for (int j = 0; j < 4; ++j) v[j] = q_rel + 16 * j < lim_rel ? __ldg(src + j) : make_uint4(0, 0, 0, 0);
                }
                const int ia = min(max(sa_rel - q_rel, 0), 64), ib = min(max(he_rel - q_rel, 0), 64);   // its bytes [ia, ib) belong to the piece
                const int64_t ib64 = -(yb + q_rel);                              // first body byte of the record in this lane
                const int ibody = ib64 <= 0 ? 0 : (ib64 >= 64 ? 64 : (int)ib64);
                const int i1 = max(ia, ibody);                                   // first body byte of the piece in this lane
                const bool act = i1 < ib;
                // keep mask and kept-base index from the closed form
                unsigned long long range = 0ull, Kp = 0ull;
                bool col0 = false;                                               // the piece's first body byte in this lane starts a line
                u = 0;
                int tnl = 64;                                             // tnl: lane index of the first predicted newline
                if (act) {
                    range = (i1 == 0 && ib == 64) ? ~0ull : (from_pos(i1) & ~from_pos(ib));
                    const uint32_t y1 = (uint32_t)(yb + q_rel + i1);             // body index of byte i1
                    const uint32_t c = col_p + (y1 - y_p);                       // column counted from the piece's first line
                    const uint32_t q = dmul ? __umulhi(c, dmul) : (uint32_t)(c >= d);
                    const int32_t col = (int32_t)(c - q * d);
                    Kp = range;
                    const uint32_t t0 = (uint32_t)i1 + ((uint32_t)W - (uint32_t)col);
                    if (t0 < (uint32_t)ib) {
                        tnl = (int)t0;
                        for (uint32_t t = t0; t < (uint32_t)ib; t += d) Kp &= ~bit_at((int)t);
                    }
                    col0 = col == 0;
                    u = (int)(q * (uint32_t)W) + col - (int)col_p;
                }
                // classification (as encode_v5.cuh): 2-bit codes and, per byte, d == 0 <=> one of ACGTacgt
                uint32_t C[4], dd[16];
                {
                    const uint32_t *xw = reinterpret_cast<const uint32_t *>(v);
                    uint32_t cb[16];
#pragma unroll
                    for (int j = 0; j < 16; ++j) {
                        const uint32_t x = xw[j];
                        cb[j] = (x & 0x06060606u) * 0x00820820u;
                        const uint32_t m = (x >> 2) & ~(x >> 1) & 0x01010101u;       // 1 where the byte has the T pattern
                        dd[j] = (x & 0xD9D9D9D9u) ^ (m * 0x0fu + 0x41414141u);       // expected masked byte: 0x41, or 0x50 for T
                    }
#pragma unroll
                    for (int h = 0; h < 4; ++h) {
                        const uint32_t lo2 = __byte_perm(cb[4 * h], cb[4 * h + 1], 0x0073);
                        const uint32_t hi2 = __byte_perm(cb[4 * h + 2], cb[4 * h + 3], 0x0073);
                        const uint32_t y = __brev(__byte_perm(lo2, hi2, 0x5410));
                        C[h] = ((y & 0x55555555u) << 1) | (((y >> 1) ^ y) & 0x55555555u);
                    }
                }
                // the layout check: the body's SKIP bytes are exactly the predicted newlines, no line starts with '>'
                const unsigned long long pd = range & ~Kp;
                unsigned long long bad = 0ull;
                bool ok = false;
                if (P.fast_lut && nl_skips && range == ~0ull && (pd & (pd - 1ull)) == 0ull) {
                    // the usual lane of wrapped FASTA: 64 body bytes, at most one predicted line end.  No per-byte flags: the
                    // three 16-byte groups without the line end must be all ACGT, the fourth all ACGT but for that byte,
                    // which must be '\n'
                    const uint32_t a0 = dd[0] | dd[1] | dd[2] | dd[3], a1 = dd[4] | dd[5] | dd[6] | dd[7];
                    const uint32_t a2 = dd[8] | dd[9] | dd[10] | dd[11], a3 = dd[12] | dd[13] | dd[14] | dd[15];
                    const int gsel = tnl >> 4;                                   // 4: no line end in this lane
                    const uint32_t other = (gsel == 0 ? 0u : a0) | (gsel == 1 ? 0u : a1) | (gsel == 2 ? 0u : a2) | (gsel == 3 ? 0u : a3);
                    if (other == 0u) {
                        if (gsel < 4) {
                            uint32_t s0 = gsel == 0 ? dd[0] : (gsel == 1 ? dd[4] : (gsel == 2 ? dd[8] : dd[12]));
                            uint32_t s1 = gsel == 0 ? dd[1] : (gsel == 1 ? dd[5] : (gsel == 2 ? dd[9] : dd[13]));
                            uint32_t s2 = gsel == 0 ? dd[2] : (gsel == 1 ? dd[6] : (gsel == 2 ? dd[10] : dd[14]));
                            uint32_t s3 = gsel == 0 ? dd[3] : (gsel == 1 ? dd[7] : (gsel == 2 ? dd[11] : dd[15]));
                            const int wi = (tnl >> 2) & 3;
                            const uint32_t bm = ~(0xffu << (8 * (tnl & 3)));
                            s0 &= wi == 0 ? bm : 0xffffffffu; s1 &= wi == 1 ? bm : 0xffffffffu;
                            s2 &= wi == 2 ? bm : 0xffffffffu; s3 &= wi == 3 ? bm : 0xffffffffu;
                            ok = (s0 | s1 | s2 | s3) == 0u && __ldg(tb + q_rel + tnl) == '\n';
                        } else ok = true;
                    }
                }
                if (!ok) {
                    // any other lane: per-byte flags, the flagged bytes through the table (what the check needs, and the class of
                    // the kept ones)
                    unsigned long long E;
                    {
                        const uint32_t *xw = reinterpret_cast<const uint32_t *>(v);
                        uint32_t fb[16];
#pragma unroll
                        for (int j = 0; j < 16; ++j) fb[j] = (((dd[j] & 0x7f7f7f7fu) + 0x7f7f7f7fu) | dd[j]) & 0x80808080u;
                        E = flags_to_plane(fb);
                        (void)xw;
                    }
                    if (!P.fast_lut) E = ~0ull;
                    E &= range;                                                  // header bytes and bytes of other records do not count
                    bad = E;
                    if (P.fast_lut && P.fast_n && __popcll(E) >= 4) E &= ~n_plane(v[0], v[1], v[2], v[3]);
                    unsigned long long skip = 0, nl = 0, gt = 0;
                    const uint8_t *vb = tb + q_rel;
                    unsigned long long rem = E;
                    while (rem) {
                        const int q = __clzll((long long)rem);
                        const unsigned long long bq = bit_at(q);
                        rem ^= bq;
                        const uint32_t byte = (uint32_t)__ldg(vb + q);
                        const uint32_t cl = sm.lut[byte];
                        if (byte == '\n') nl |= bq;
                        if (byte == '>') gt |= bq;
                        if (cl == CLS_SKIP) skip |= bq;
                        else if (Kp & bq) {
                            if (cl < CLS_N) bad &= ~bq;
                            v7::set_digit(C, q, cl < CLS_N ? cl : (cl == CLS_N ? 2u : 1u));
                        }
                    }
                    unsigned long long lstart = (pd >> 1) & range;               // a line starts behind every predicted newline
                    if (col0) lstart |= bit_at(i1);
                    ok = skip == pd && (pd & ~nl) == 0ull && (!P.strip_headers || (gt & lstart) == 0ull);
                }
                if (!ok) irregular = true;
                // compaction in registers
                const unsigned long long keep = Kp;
                const int n = __popcll(keep);
                if (n == 0) { C[0] = C[1] = C[2] = C[3] = 0u; bad = 0ull; }
                else if (n == 63) v7::delete_one(C, bad, __clzll((long long)~keep));
                else if (n != 64) v7::delete_runs(C, bad, keep);
                const uint32_t Fw[2] = {(uint32_t)(bad >> 32), (uint32_t)bad};
                if (__any_sync(FULL, bad != 0ull)) has_flags = true;             // (warp-uniform) the piece holds flagged bases
                // append at the closed-form position u
                if (__all_sync(FULL, n >= 32)) {
                    // every lane fills a whole word: interior words are written once (a lane's last partial word travels to the
                    // next lane by shuffle); the chunk's first and last word are shared with its neighbours and OR-ed in
                    {
                        const int cw0 = u >> 4, csh = 2 * (u & 15), cend = csh + 2 * n;      // cend in [64, 158]
                        const uint32_t w0 = C[0] >> csh, w1 = __funnelshift_r(C[1], C[0], csh), w2 = __funnelshift_r(C[2], C[1], csh),
                                       w3 = __funnelshift_r(C[3], C[2], csh), w4 = __funnelshift_r(0u, C[3], csh);
                        const int li = cend >> 5;                                            // 2, 3 or 4
                        uint32_t part = li == 2 ? w2 : (li == 3 ? w3 : w4);
                        if ((cend & 31) == 0) part = 0u;
                        const uint32_t prev = __shfl_up_sync(FULL, part, 1);
                        if (lane == 0) { if (w0) atomicOr(&cw[cw0], w0); } else cw[cw0] = w0 | prev;
                        cw[cw0 + 1] = w1;
                        if (cend >= 96) cw[cw0 + 2] = w2;
                        if (cend >= 128) cw[cw0 + 3] = w3;
                        if (lane == 31 && part) atomicOr(&cw[cw0 + li], part);
                    }
                    {
                        const int fw0 = u >> 5, fsh = u & 31, fend = fsh + n;                // fend in [32, 95]
                        const uint32_t w0 = Fw[0] >> fsh, w1 = __funnelshift_r(Fw[1], Fw[0], fsh), w2 = __funnelshift_r(0u, Fw[1], fsh);
                        const int li = fend >> 5;                                            // 1 or 2
                        uint32_t part = li == 1 ? w1 : w2;
                        if ((fend & 31) == 0) part = 0u;
                        const uint32_t prev = __shfl_up_sync(FULL, part, 1);
                        if (lane == 0) { if (w0) atomicOr(&fw[fw0], w0); } else fw[fw0] = w0 | prev;
                        if (fend >= 64) fw[fw0 + 1] = w1;
                        if (lane == 31 && part) atomicOr(&fw[fw0 + li], part);
                    }
                } else if (n > 0) {
                    const int cw0 = u >> 4, csh = 2 * (u & 15), cend = csh + 2 * n;
                    uint32_t cwv[5];
                    cwv[0] = C[0] >> csh;
                    cwv[1] = __funnelshift_r(C[1], C[0], csh);
                    cwv[2] = __funnelshift_r(C[2], C[1], csh);
                    cwv[3] = __funnelshift_r(C[3], C[2], csh);
                    cwv[4] = __funnelshift_r(0u, C[3], csh);
#pragma unroll
                    for (int i = 0; i < 5; ++i)
                        if (32 * i < cend && cwv[i]) atomicOr(&cw[cw0 + i], cwv[i]);
                    const int fw0 = u >> 5, fsh = u & 31, fend = fsh + n;
                    uint32_t bwv[3];
                    bwv[0] = Fw[0] >> fsh; bwv[1] = __funnelshift_r(Fw[1], Fw[0], fsh); bwv[2] = __funnelshift_r(0u, Fw[1], fsh);
#pragma unroll
                    for (int i = 0; i < 3; ++i)
                        if (32 * i < fend && bwv[i]) atomicOr(&fw[fw0 + i], bwv[i]);
                }
            }
            __syncwarp();
            // ---- tokens whose first base lies in the piece: record base K0 + i sits at stream position i ---------------------
            // windows j of the record with K0 <= j k < K0 + nK, as piece-relative first bases u = j k - K0
            const uint32_t jfirst = (K0 + (uint32_t)k - 1u) / (uint32_t)k;       // first window of the record that starts in the piece
            const int ufirst = (int)(jfirst * (uint32_t)k - K0);                 //   and the stream position of its first base
            int nwp = ufirst < nK ? (int)((uint32_t)(nK - ufirst + k - 1) / (uint32_t)k) : 0;   // windows that start in the piece
            if (nwin != FAR && jfirst + (uint32_t)nwp > nwin) nwp = nwin > jfirst ? (int)(nwin - jfirst) : 0;
            if (FUSED && jfirst + (uint32_t)nwp > jcap) nwp = jcap > jfirst ? (int)(jcap - jfirst) : 0;
            const int64_t g0 = g_base + jfirst;                                  // destination index of the first of them
            IdT *const idp = ids + g0;
            int xa = nwp, xb = nwp;                                              // windows [xa, xb) go through the 16-byte group cutter
            if (vec_ok) {
                xa = (int)((R - (g0 & (R - 1))) & (R - 1));
                xb = xa + ((nwp - xa) & ~(R - 1));
                if (g0 + xb > A.ids_cap) xb = xa;
                if (nwp < xa || xb <= xa) { xa = nwp; xb = nwp; }
            }
            for (int x = xa + lane * R; x < xb; x += 32 * R)
                emit_group_sel<IdT, KK>(A, cw, fw, ufirst + x * k, idp + x, affine, kk, has_flags);
            {
                // the windows in front of and behind the groups, one per lane
                const int n1 = xa, n2 = nwp - xb;
                for (int y = lane; y < n1 + n2; y += 32) {
                    const int x = y < n1 ? y : xb + (y - n1);
                    store_id<IdT>(A, g0 + x, w_window_id(P, cw, fw, ufirst + x * k));
                }
            }
            if (P.mode == MODE_KMER && n_r != FAR) {
                // the n mod k trailing bases of the record, if they lie in the piece
                const int64_t tb0 = (int64_t)nwin * k;
                if (P.tail_policy == TAIL_PER_BASE) {
                    const int64_t b0 = K0 > tb0 ? K0 : tb0, b1 = (int64_t)K0 + nK < n_r ? (int64_t)K0 + nK : n_r;
                    for (int64_t bb = b0 + lane; bb < b1; bb += 32) {
                        const uint32_t c = w_class(cw, fw, (int)(bb - K0));
                        const int32_t id = c <= CLS_N ? (P.remap4 ? P.nt_ids[c] : (int32_t)(P.base_id + P.four_k + c)) : P.unk_id;
                        if (!FUSED || nwin + (uint32_t)(bb - tb0) < jcap) store_id<IdT>(A, g_base + nwin + (bb - tb0), id);
                    }
                } else if (P.tail_policy == TAIL_UNK) {
                    if (lane == 0 && n_r > tb0 && tb0 >= K0 && tb0 < K0 + nK && (!FUSED || nwin < jcap)) store_id<IdT>(A, g_base + nwin, P.unk_id);
                }
            }
            __syncwarp();
        }
        if (__any_sync(FULL, irregular)) break;                     // published below; the other warps stop at their next tile
        tile = next_tile;
    }
    if (__any_sync(FULL, irregular) && lane == 0) *F.irregular = 1u;
}

}  // namespace fa
}  // namespace dtk
