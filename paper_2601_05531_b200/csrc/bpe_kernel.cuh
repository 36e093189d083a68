// bpe_kernel.cuh -- BPE merges, organised around ACGT SEGMENTS, lowest rank first.
//
// Semantics: the kept classes of a read are cut at every N / UNK (each is its own token
// and a hard boundary); inside each ACGT segment, repeat { take the lowest-rank adjacent pair that has a rule; replace
// all its occurrences left to right without overlap } until no adjacent pair has a rule.  For a valid table (rule r's
// parts are tokens < 4 + r) this equals applying ONE occurrence at a time in (rank, position) order: a merge of rank m
// only creates pairs of rank > m, so the minimum never decreases and equal ranks are met left to right.  That is the
// form used here.
//
// Passes (all stream-ordered, no host synchronisation):
//   bpe_segments_kernel<false>  one warp per read: finds the ACGT segments (ballots over 32 classes at a time) and
//                               counts them per LENGTH BIN (width 8 up to 512 symbols)
//   bpe_bins_kernel             66 threads: bin -> first slot in the segment list / first work item, longest bins first
//   bpe_segments_kernel<true>   finds them again, writes the sorted segment list; writes the N / UNK tokens and the
//                               single-base segments to tmp_tok, holes elsewhere; per-read token counts of those
//   bpe_merge_kernel            persistent warps take work items from an atomic counter, longest segments first:
//                               one segment per LANE (2..64 symbols), per 2, 4, 8 LANES (up to 128, 256, 512) or per WARP
//                               (513..2048).
//                               Lanes of a warp work on segments of one bin, i.e. of nearly equal length.
//                               Symbols and cached pair ranks sit in the warp's shared-memory slice, one 32-bit word per
//                               position (rank << 16 | symbol), interleaved so that the lanes hit different banks.
//                               A round = min over (rank, position) of the alive pairs, one merge: the right symbol dies
//                               in place (no compaction), two rule look-ups refresh the ranks of the pairs that touch
//                               the new token.  No block barrier anywhere; a segment is finished when ITS minimum is
//                               "no rule".
//   bpe_merge_giant_kernel      the same code, one warp per CTA with a large slice, for segments over 2048 symbols
//   scan_counts_kernel, bpe_gather_kernel   token counts -> out_offsets; tokens of tmp_tok -> ids
#pragma once
#include "common.cuh"

namespace dtk {

constexpr uint32_t BPE_INF = 0xffffu;          // "no rule" rank / also the largest uint16
constexpr uint32_t SYM_N = 0xffffu, SYM_UNK = 0xfffeu;   // boundary symbols (never merged, never removed)
constexpr uint64_t HASH_EMPTY = ~0ull;
constexpr uint32_t SYM_HOLE = 0xfffdu;          // tmp_tok entry that holds no token (the gather kernel drops it);
                                                //   in the merge workspace: a symbol that was merged into its left neighbour

constexpr int BPE_NB = 66;                      // length bins: 0..63 = 8 lengths each (2..512), 64 = 513..2048, 65 = longer
constexpr int BPE_MAIN_BINS = 65;               // bins the main merge kernel serves
constexpr int BPE_SLOT_WORDS = 2048;            // shared-memory words per warp of the main merge kernel
constexpr int BPE_WARPS = 8;                    // warps per CTA of the main merge kernel
constexpr int BPE_GIANT_MAX = 49152;            // symbols the giant kernel's slice can hold at most (192 KiB)
constexpr int BPE_SEG_WARPS = 8;                // warps (= reads in flight) per CTA of the segment finder

struct BpeSeg { uint32_t start, len, read, pad; };   // start: index into cls / tmp_tok of the segment's first symbol

__host__ __device__ __forceinline__ int bpe_bin(uint32_t len) { return len <= 512u ? (int)((len - 1u) >> 3) : (len <= (uint32_t)BPE_SLOT_WORDS ? 64 : 65); }
// lanes per segment: G lanes share BPE_SLOT_WORDS / (32 / G) positions -- 64 per lane
__host__ __device__ __forceinline__ int bpe_bin_lanes(int bin) { return bin < 8 ? 1 : (bin < 16 ? 2 : (bin < 32 ? 4 : (bin < 64 ? 8 : 32))); }
// processing order: longest first (bin 64, 63, ..., 0), the giant bin last (its own kernel)
__host__ __device__ __forceinline__ int bpe_ord(int bin) { return bin == 65 ? 65 : 64 - bin; }

struct BpeArgs {
    const uint8_t *cls;            // compact kept classes of all reads (class pass output)
    const int64_t *koff;           // [n_rec + 1] kept-base CSR offsets (class pass output)
    int64_t n_rec;
    const uint64_t *table;         // open-addressing hash: (left<<16|right)<<32 | rank
    uint32_t table_mask;
    uint16_t *tmp_tok;             // per kept base: a token of the segment that started there, or SYM_HOLE
    int32_t *tok_cnt;              // [n_rec] tokens per read
    uint32_t *status;
    BpeSeg *segs;                  // segment list, sorted by bin in processing order
    int64_t segs_cap;
    uint32_t *ctl;                 // control block (zeroed before every call): see the CTL_* offsets
    uint32_t *cta_hist;            // [CTAs of the segment finder][BPE_NB] segments per bin of each CTA's reads (count pass -> fill pass)
    int32_t giant_cap;             // symbols the giant kernel's slice holds
};
// control block layout (uint32 words)
constexpr int CTL_CNT = 0;                      // [BPE_NB] segments per bin
constexpr int CTL_FILL = CTL_CNT + BPE_NB;      // [BPE_NB] fill cursors
constexpr int CTL_BASE = CTL_FILL + BPE_NB;     // [BPE_NB + 1] by processing order: first slot in segs
constexpr int CTL_ITEM = CTL_BASE + BPE_NB + 1; // [BPE_NB + 1] by processing order: first work item
constexpr int CTL_CTR = CTL_ITEM + BPE_NB + 1;  // [2] work-item counters: main, giant
constexpr int CTL_WORDS = CTL_CTR + 2;

__device__ __forceinline__ uint32_t bpe_hash(uint32_t key) {
    key ^= key >> 15; key *= 0x2c1b3c6du; key ^= key >> 12; key *= 0x297a2d39u; key ^= key >> 15;
    return key;
}

__device__ __forceinline__ uint32_t bpe_rank(const BpeArgs &A, uint32_t l, uint32_t r) {
    const uint32_t key = (l << 16) | r;
    uint32_t h = bpe_hash(key) & A.table_mask;
    for (;;) {
        const uint64_t s = __ldg(A.table + h);
        if (s == HASH_EMPTY) return BPE_INF;
        if ((uint32_t)(s >> 32) == key) return (uint32_t)s;
        h = (h + 1) & A.table_mask;
    }
}

// ---- segment finder ----------------------------------------------------------------------------------------
// One warp per read, 32 classes per step.  FILL = false: counts the segments of 2 or more symbols per length bin.
// FILL = true: writes their records into the bin-sorted list, the tokens that need no merging (N, UNK, single bases) to
// tmp_tok with holes everywhere else, and the number of those tokens to tok_cnt.
template <bool FILL>
__global__ void __launch_bounds__(BPE_SEG_WARPS * 32) bpe_segments_kernel(const __grid_constant__ BpeArgs A) {
    constexpr uint32_t FULL = 0xffffffffu;
    __shared__ uint32_t hist[BPE_NB];           // segments of this CTA's reads per bin, then the fill cursor inside the CTA's range
    __shared__ uint32_t first[BPE_NB];          // FILL: first slot of the CTA's range in each bin
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int64_t r = (int64_t)blockIdx.x * BPE_SEG_WARPS + warp;
    for (int i = tid; i < BPE_NB; i += blockDim.x) hist[i] = 0u;
    __syncthreads();
    const bool have = r < A.n_rec;
    const int64_t k0 = have ? A.koff[r] : 0;
    const int n = have ? (int)(A.koff[r + 1] - k0) : 0;

    // sweep(emit): calls emit(start, len) once per segment (start relative to the read), from one lane.  With FILL it also
    // writes the tokens that need no merging (N, UNK) and holes everywhere else, before the emits of the same step.
    int direct = 0;
    auto sweep = [&](auto &&emit) {
        int open = -1;                          // start of the segment still open at the end of the previous step
        for (int base = 0; base < n; base += 32) {
            const int i = base + lane;
            const uint32_t c = i < n ? A.cls[k0 + i] : 255u;
            if (FILL) {
                if (i < n) {
                    A.tmp_tok[k0 + i] = (uint16_t)(c < CLS_N ? SYM_HOLE : (c == CLS_N ? SYM_N : SYM_UNK));
                    direct += c >= CLS_N;
                }
                __syncwarp();
            }
            const uint32_t bm = __ballot_sync(FULL, c >= CLS_N);          // boundaries (positions past the end count as one)
            const bool prevb = lane ? ((bm >> (lane - 1)) & 1u) : (open < 0);
            const bool st = c < CLS_N && prevb;                           // a segment starts here
            if (open >= 0 && bm && lane == 0) emit(open, base + __ffs(bm) - 1 - open);
            const uint32_t above = lane == 31 ? 0u : (bm & (FULL << (lane + 1)));
            if (st && above) emit(i, base + __ffs(above) - 1 - i);
            if (bm == 0u) { if (open < 0) open = base; }
            else { const int lastb = 31 - __clz(bm); open = lastb < 31 ? base + lastb + 1 : -1; }
        }
        if (open >= 0 && lane == 0) emit(open, n - open);                 // (n is a multiple of 32 and the read ends open)
    };

    if (!FILL) {
        sweep([&](int, int len) { if (len >= 2 && len <= A.giant_cap) atomicAdd(&hist[bpe_bin((uint32_t)len)], 1u); });
        __syncthreads();
        for (int i = tid; i < BPE_NB; i += blockDim.x) {
            const uint32_t c = hist[i];
            A.cta_hist[(size_t)blockIdx.x * BPE_NB + i] = c;
            if (c) atomicAdd(&A.ctl[CTL_CNT + i], c);
        }
        return;
    }
    // the CTA's range in every bin of the list
    for (int i = tid; i < BPE_NB; i += blockDim.x) {
        const uint32_t c = A.cta_hist[(size_t)blockIdx.x * BPE_NB + i];
        first[i] = c ? A.ctl[CTL_BASE + bpe_ord(i)] + atomicAdd(&A.ctl[CTL_FILL + i], c) : 0u;
    }
    __syncthreads();
    sweep([&](int start, int len) {
        if (len == 1) { A.tmp_tok[k0 + start] = (uint16_t)A.cls[k0 + start]; ++direct; return; }
        const int bin = bpe_bin((uint32_t)len);
        if (len > A.giant_cap) { A.status[0] = 1u; return; }               // does not fit any workspace: reported, no tokens
        const uint32_t slot = first[bin] + atomicAdd(&hist[bin], 1u);
        if ((int64_t)slot < A.segs_cap) A.segs[slot] = BpeSeg{(uint32_t)(k0 + start), (uint32_t)len, (uint32_t)r, 0u};
        else A.status[0] = 1u;
    });
    direct = __reduce_add_sync(FULL, direct);
    if (have && lane == 0) A.tok_cnt[r] = direct;
}

// bin counts -> list slots and work items, in processing order
__global__ void __launch_bounds__(128) bpe_bins_kernel(const __grid_constant__ BpeArgs A) {
    __shared__ uint32_t cnt[BPE_NB], items[BPE_NB];
    const int o = threadIdx.x;                  // processing-order index
    if (o < BPE_NB) {
        const int bin = o == 65 ? 65 : 64 - o;
        const uint32_t c = A.ctl[CTL_CNT + bin];
        cnt[o] = c;
        const uint32_t per = 32u / (uint32_t)bpe_bin_lanes(bin);          // segments per work item
        items[o] = (c + per - 1u) / per;
    }
    __syncthreads();
    if (o == 0) {
        uint32_t s = 0, t = 0;
        for (int i = 0; i < BPE_NB; ++i) {
            A.ctl[CTL_BASE + i] = s; A.ctl[CTL_ITEM + i] = t;
            s += cnt[i]; t += items[i];
        }
        A.ctl[CTL_BASE + BPE_NB] = s; A.ctl[CTL_ITEM + BPE_NB] = t;
    }
}

// ---- the merge loop: G lanes per segment, 32 / G segments per warp ------------------------------------------------
// slice: the warp's shared-memory words; position i of the warp's group q sits at slice[i * (32 / G) + q].
template <int G>
__device__ __forceinline__ void bpe_merge_item(const BpeArgs &A, uint32_t *slice, uint32_t seg_lo, uint32_t seg_hi, int lane) {
    constexpr uint32_t FULL = 0xffffffffu;
    constexpr int NG = 32 / G;
    const int q = lane / G, g = lane % G;
    const uint32_t si = seg_lo + (uint32_t)q;
    const bool have = si < seg_hi;
    BpeSeg sg = BpeSeg{0u, 0u, 0u, 0u};
    if (have) sg = A.segs[si];
    const int L = (int)sg.len;
    uint32_t *w = slice + q;
    // symbols, then the rank of every adjacent pair
    for (int i = g; i < L; i += G) w[i * NG] = (BPE_INF << 16) | (uint32_t)A.cls[sg.start + i];
    if (G > 1) __syncwarp();
    for (int i = g; i + 1 < L; i += G) {
        const uint32_t s0 = w[i * NG] & 0xffffu, s1 = w[(i + 1) * NG] & 0xffffu;
        w[i * NG] = (bpe_rank(A, s0, s1) << 16) | s0;
    }
    if (G > 1) __syncwarp();
    bool done = L < 2;
    for (;;) {
        // lowest (rank, position) over the segment's alive pairs
        uint32_t key = 0xffffffffu;
        if (!done) {
            int i = g;
#pragma unroll 4
            for (; i < L; i += G) key = min(key, (w[i * NG] & 0xffff0000u) | (uint32_t)i);
        }
#pragma unroll
        for (int d = G >> 1; d > 0; d >>= 1) key = min(key, __shfl_xor_sync(FULL, key, d));
        if ((key >> 16) == BPE_INF) done = true;
        if (__all_sync(FULL, done)) break;
        if (!done) {
            const uint32_t m = key >> 16;
            const int bi = (int)(key & 0xffffu);
            // alive neighbours: four candidate positions are loaded at a time (dead runs are a few symbols long)
            auto next_alive = [&](int from) {                 // first alive position >= from, or L
                for (int b0 = from; b0 < L; b0 += 4) {
                    uint32_t s4[4];
#pragma unroll
                    for (int x = 0; x < 4; ++x) s4[x] = w[min(b0 + x, L - 1) * NG] & 0xffffu;
#pragma unroll
                    for (int x = 0; x < 4; ++x) if (b0 + x < L && s4[x] != SYM_HOLE) return b0 + x;
                }
                return L;
            };
            const int j = next_alive(bi + 1);                 // the pair's right symbol (it exists)
            const int jn = next_alive(j + 1);                 // the alive symbol behind it, if any
            int p = bi - 1;                                   // the alive symbol in front, if any
            for (; p >= 0; p -= 4) {
                uint32_t s4[4];
#pragma unroll
                for (int x = 0; x < 4; ++x) s4[x] = w[max(p - x, 0) * NG] & 0xffffu;
                int f = -1;
#pragma unroll
                for (int x = 3; x >= 0; --x) if (p - x >= 0 && s4[x] != SYM_HOLE) f = p - x;
                if (f >= 0) { p = f; break; }
            }
            if (p < 0) p = -1;
            const uint32_t ns = 4u + m;
            if (g == 0) {
                const uint32_t r1 = jn < L ? bpe_rank(A, ns, w[jn * NG] & 0xffffu) : BPE_INF;
                w[bi * NG] = (r1 << 16) | ns;
                w[j * NG] = (BPE_INF << 16) | SYM_HOLE;
            }
            if (g == (G > 1 ? 1 : 0) && p >= 0) {
                const uint32_t sp = w[p * NG] & 0xffffu;
                w[p * NG] = (bpe_rank(A, sp, ns) << 16) | sp;
            }
        }
        if (G > 1) __syncwarp();
    }
    // tokens of the segment, in order, at the segment's own place
    if (have && g == 0) {
        int cnt = 0;
        for (int i = 0; i < L; ++i) {
            const uint32_t s = w[i * NG] & 0xffffu;
            if (s != SYM_HOLE) A.tmp_tok[sg.start + cnt++] = (uint16_t)s;
        }
        atomicAdd(&A.tok_cnt[sg.read], cnt);
    }
}

__global__ void __launch_bounds__(BPE_WARPS * 32) bpe_merge_kernel(const __grid_constant__ BpeArgs A) {
    extern __shared__ __align__(16) uint32_t bpe_smem[];
    constexpr uint32_t FULL = 0xffffffffu;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    uint32_t *slice = bpe_smem + warp * BPE_SLOT_WORDS;
    // work-item table (processing order), three entries per lane
    uint32_t ib[3];
#pragma unroll
    for (int x = 0; x < 3; ++x) { const int o = lane + 32 * x; ib[x] = o <= BPE_MAIN_BINS ? A.ctl[CTL_ITEM + o] : 0xffffffffu; }
    const uint32_t n_items = A.ctl[CTL_ITEM + BPE_MAIN_BINS];
    for (;;) {
        uint32_t t = 0;
        if (lane == 0) t = atomicAdd(&A.ctl[CTL_CTR], 1u);
        t = __shfl_sync(FULL, t, 0);
        if (t >= n_items) break;
        // o = last processing-order index whose first item is <= t
        int o = 0;
#pragma unroll
        for (int x = 0; x < 3; ++x) o += __popc(__ballot_sync(FULL, ib[x] <= t));
        o -= 1;
        // (empty bins share their first item with the next one: the last such index is the bin that owns item t)
        const int bin = 64 - o;
        const int G = bpe_bin_lanes(bin);
        const uint32_t lo = A.ctl[CTL_BASE + o] + (t - A.ctl[CTL_ITEM + o]) * (uint32_t)(32 / G);
        const uint32_t hi = A.ctl[CTL_BASE + o + 1];
        if (G == 1) bpe_merge_item<1>(A, slice, lo, hi, lane);
        else if (G == 2) bpe_merge_item<2>(A, slice, lo, hi, lane);
        else if (G == 4) bpe_merge_item<4>(A, slice, lo, hi, lane);
        else if (G == 8) bpe_merge_item<8>(A, slice, lo, hi, lane);
        else bpe_merge_item<32>(A, slice, lo, hi, lane);
        __syncwarp();
    }
}

// segments over BPE_SLOT_WORDS symbols: one warp per CTA, the whole dynamic shared memory is its slice
__global__ void __launch_bounds__(32) bpe_merge_giant_kernel(const __grid_constant__ BpeArgs A) {
    extern __shared__ __align__(16) uint32_t bpe_smem[];
    constexpr uint32_t FULL = 0xffffffffu;
    const int lane = threadIdx.x;
    const uint32_t lo = A.ctl[CTL_BASE + 65], hi = A.ctl[CTL_BASE + 66];
    for (;;) {
        uint32_t t = 0;
        if (lane == 0) t = atomicAdd(&A.ctl[CTL_CTR + 1], 1u);
        t = __shfl_sync(FULL, t, 0);
        if (lo + t >= hi) break;
        bpe_merge_item<32>(A, bpe_smem, lo + t, hi, lane);
        __syncwarp();
    }
}

// single-block exclusive scan of per-read token counts -> out_offsets (int64), total in the last entry; four counts per
// thread per step
__global__ void __launch_bounds__(1024) scan_counts_kernel(const int32_t *cnt, int64_t n, int64_t *out_off) {
    __shared__ long long wsum[32];
    __shared__ long long s_carry;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (tid == 0) s_carry = 0;
    __syncthreads();
    for (int64_t base = 0; base < n; base += 4096) {
        const int64_t i = base + 4 * (int64_t)tid;
        int v[4];
#pragma unroll
        for (int x = 0; x < 4; ++x) v[x] = (i + x < n) ? cnt[i + x] : 0;
        const long long mine = (long long)v[0] + v[1] + v[2] + v[3];
        long long inc = mine;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) { long long t = __shfl_up_sync(0xffffffffu, inc, d); if (lane >= d) inc += t; }
        if (lane == 31) wsum[warp] = inc;
        __syncthreads();
        long long woff = 0, tot = 0;
        for (int w = 0; w < 32; ++w) { long long t = wsum[w]; if (w < warp) woff += t; tot += t; }
        long long run = s_carry + woff + inc - mine;
#pragma unroll
        for (int x = 0; x < 4; ++x) { if (i + x < n) out_off[i + x] = run; run += v[x]; }
        __syncthreads();
        if (tid == 0) s_carry += tot;
        __syncthreads();
    }
    if (tid == 0) out_off[n] = s_carry;
}

// ids of read r = its tmp_tok entries that are not holes, in order (one warp per read)
template <typename IdT>
__global__ void __launch_bounds__(256) bpe_gather_kernel(const uint16_t *tmp_tok, const int64_t *koff,
                                                         const int64_t *out_off, int64_t n_rec, IdT *ids,
                                                         int64_t ids_cap, int32_t base_id, int32_t n_id,
                                                         int32_t unk_id, uint32_t *status) {
    constexpr uint32_t FULL = 0xffffffffu;
    const int lane = threadIdx.x & 31;
    const int64_t warp = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int64_t nwarps = ((int64_t)gridDim.x * blockDim.x) >> 5;
    for (int64_t r = warp; r < n_rec; r += nwarps) {
        const int64_t k0 = koff[r], o_end = out_off[r + 1];
        const int n = (int)(koff[r + 1] - k0);
        int64_t o = out_off[r];
        for (int base = 0; base < n && o < o_end; base += 32) {
            const int i = base + lane;
            const uint32_t s = i < n ? (uint32_t)tmp_tok[k0 + i] : SYM_HOLE;
            const uint32_t vm = __ballot_sync(FULL, s != SYM_HOLE);
            const int64_t at = o + __popc(vm & ((1u << lane) - 1u));
            if (s != SYM_HOLE && at < o_end) {               // (a segment that did not fit the workspace has no tokens)
                const int32_t id = s == SYM_N ? n_id : (s == SYM_UNK ? unk_id : (int32_t)(base_id + s));
                if (at < ids_cap) ids[at] = (IdT)id; else status[0] = 1u;
            }
            o += __popc(vm);
        }
    }
}

}  // namespace dtk
