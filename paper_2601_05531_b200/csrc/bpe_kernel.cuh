// bpe_kernel.cuh -- BPE merge kernel: one read per thread block, lowest rank first.
//
// Semantics: the kept classes of a read are cut at every
// N / UNK (each is its own token and a hard boundary); inside each ACGT segment, repeat
// { take the lowest-rank adjacent pair that has a rule; replace all its occurrences left to
// right without overlap } until no adjacent pair has a rule.
//
// Parallel form: all segments of the read advance together, one "round" per iteration; in a
// round every segment applies ITS OWN current minimum rank (segments never interact, so this
// equals the sequential order segment by segment).  Merging every locally-minimal pair at once
// would be wrong (SURVEY.md section 7 hard part 5), so only pairs whose rank equals the
// segment minimum fire.  Pair ranks are cached next to the symbols and only pairs touching a
// freshly merged token are looked up again (one hash probe sequence each).
#pragma once
#include "common.cuh"

namespace dtk {

constexpr int BPE_NT = 256;
constexpr uint32_t BPE_INF = 0xffffu;          // "no rule" rank / also the largest uint16
constexpr uint32_t SYM_N = 0xffffu, SYM_UNK = 0xfffeu;   // boundary symbols (never merged, never removed)
constexpr uint64_t HASH_EMPTY = ~0ull;
constexpr uint32_t SYM_HOLE = 0xfffdu;          // tmp_tok entry that holds no token (the gather kernel drops it)

struct BpeArgs {
    const uint8_t *cls;            // compact kept classes of all reads (pass A output)
    const int64_t *koff;           // [n_rec + 1] kept-base CSR offsets (pass A output)
    int64_t n_rec;
    const uint64_t *table;         // open-addressing hash: (left<<16|right)<<32 | rank
    uint32_t table_mask;
    int32_t cap;                   // symbols per read the shared-memory workspace can hold
    uint16_t *tmp_tok;             // per kept base of read r: a token of the segment that started there, or SYM_HOLE
    int32_t *tok_cnt;              // [n_rec] tokens per read
    uint32_t *status;
};

__device__ __forceinline__ uint32_t bpe_hash(uint32_t key) {
    key ^= key >> 15; key *= 0x2c1b3c6du; key ^= key >> 12; key *= 0x297a2d39u; key ^= key >> 15;
    return key;
}

__device__ __forceinline__ uint32_t bpe_rank(const BpeArgs &A, uint32_t l, uint32_t r) {
    if (l >= SYM_UNK || r >= SYM_UNK) return BPE_INF;
    const uint32_t key = (l << 16) | r;
    uint32_t h = bpe_hash(key) & A.table_mask;
    for (;;) {
        uint64_t s = __ldg(A.table + h);
        if (s == HASH_EMPTY) return BPE_INF;
        if ((uint32_t)(s >> 32) == key) return (uint32_t)s;
        h = (h + 1) & A.table_mask;
    }
}

// block-wide exclusive count of a flag (BPE_NT threads), one barrier: ballot + popc inside the warp, the warp totals
// through shared memory.  Consecutive calls alternate between the two halves of warp_tmp (pp), so a warp still
// reading one half never meets the writes of the next call.
__device__ __forceinline__ int bpe_exscan(bool f, int (*warp_tmp)[BPE_NT / 32], int &pp, int &total) {
    static_assert((BPE_NT / 32) % 4 == 0, "warp totals are read four at a time");
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const uint32_t b = __ballot_sync(0xffffffffu, f);
    if (lane == 0) warp_tmp[pp][warp] = __popc(b);
    __syncthreads();
    int woff = 0, tot = 0;
#pragma unroll
    for (int q = 0; q < BPE_NT / 128; ++q) {
        const int4 t = *reinterpret_cast<const int4 *>(&warp_tmp[pp][4 * q]);
        const int v[4] = {t.x, t.y, t.z, t.w};
#pragma unroll
        for (int j = 0; j < 4; ++j) { if (4 * q + j < warp) woff += v[j]; tot += v[j]; }
    }
    pp ^= 1;
    total = tot;
    return woff + __popc(b & ((1u << lane) - 1u));
}

// minimum of rank rk into the 16-bit slot of segment sg (two slots per 32-bit word, CAS on the word)
__device__ __forceinline__ void bpe_seg_min(uint16_t *segmin, uint32_t sg, uint32_t rk) {
    uint32_t *w = reinterpret_cast<uint32_t *>(segmin) + (sg >> 1);
    uint32_t old = *w;
    for (;;) {
        const uint32_t half = (sg & 1) ? (old >> 16) : (old & 0xffffu);
        if (half <= rk) break;
        const uint32_t neu = (sg & 1) ? ((old & 0xffffu) | (rk << 16)) : ((old & 0xffff0000u) | rk);
        const uint32_t got = atomicCAS(w, old, neu);
        if (got == old) break;
        old = got;
    }
}

// ranks of one warp's 32 consecutive symbols into the per-segment minima: segments are contiguous, so a segmented
// min-scan over the warp leaves each run's minimum in its last lane, which alone touches shared memory
__device__ __forceinline__ bool bpe_warp_seg_min(uint16_t *segmin, uint32_t sg, uint32_t rk, bool valid) {
    constexpr uint32_t FULL = 0xffffffffu;
    const int lane = threadIdx.x & 31;
    if (!valid) { sg = 0xffffffffu; rk = BPE_INF; }
    uint32_t v = rk;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const uint32_t t = __shfl_up_sync(FULL, v, d), st = __shfl_up_sync(FULL, sg, d);
        if (lane >= d && st == sg) v = min(v, t);
    }
    const uint32_t nsg = __shfl_down_sync(FULL, sg, 1);
    const bool last = lane == 31 || nsg != sg;
    if (valid && last && v != BPE_INF) bpe_seg_min(segmin, sg, v);
    return __any_sync(FULL, valid && rk != BPE_INF);
}

// dynamic shared memory layout: sym[2][cap] rnk[2][cap] seg[2][cap] src[cap] segmin[2][cap+2] origin[cap]
// segstart[cap], all uint16.  A segment none of whose pairs has a rule any more is finished: the next compaction pass
// writes its tokens to tmp_tok at the segment's own place in the read (the rest of its span stays SYM_HOLE) and drops
// it from the working sequence, so late rounds only touch the few long segments that are still merging.
// One round = compaction pass (one barrier per chunk of BPE_NT symbols) -> barrier -> rank pass, which also collects
// the next round's per-segment minima into the other segmin buffer -> barrier.
__global__ void __launch_bounds__(BPE_NT) bpe_reads_kernel(const __grid_constant__ BpeArgs A) {
    extern __shared__ __align__(16) uint16_t sh[];
    __shared__ __align__(16) int warp_tmp[2][BPE_NT / 32];
    const int cap = A.cap, tid = threadIdx.x;
    uint16_t *symb[2] = {sh, sh + cap};
    uint16_t *rnkb[2] = {sh + 2 * cap, sh + 3 * cap};
    uint16_t *segb[2] = {sh + 4 * cap, sh + 5 * cap};
    uint16_t *src = sh + 6 * cap;
    uint16_t *sminb[2] = {sh + 7 * cap, sh + 8 * cap + 2};
    uint16_t *origin = sh + 9 * cap + 4;       // [cap] position in the read of each segment's first symbol
    uint16_t *segstart = sh + 10 * cap + 4;    // [cap] index in the current sequence of each segment's first symbol
    __shared__ int s_cnt;
    int pp = 0;

    for (int64_t r = blockIdx.x; r < A.n_rec; r += gridDim.x) {
        const int64_t k0 = A.koff[r];
        const int64_t n64 = A.koff[r + 1] - k0;
        __syncthreads();
        if (n64 > cap) {                      // read does not fit the workspace: report, emit nothing
            if (tid == 0) { A.status[0] = 1u; A.tok_cnt[r] = 0; }
            continue;
        }
        int n = (int)n64, cur = 0, ms = 0;
        // ---- load symbols, segment ids (a boundary symbol forms its own segment) --------
        // seg id = number of "segment starts" at or before i, minus 1; a start is i == 0, a boundary,
        // or the position right after a boundary.
        for (int i = tid; i < n; i += BPE_NT) {
            const uint32_t c = A.cls[k0 + i];
            symb[0][i] = (uint16_t)(c < CLS_N ? c : (c == CLS_N ? SYM_N : SYM_UNK));
        }
        for (int i = tid; i <= n; i += BPE_NT) sminb[0][i] = (uint16_t)BPE_INF;     // at most n segments
        for (int i = tid; i < n; i += BPE_NT) A.tmp_tok[k0 + i] = (uint16_t)SYM_HOLE;
        if (tid == 0) s_cnt = 0;
        __syncthreads();
        int seg_base = 0;
        for (int base = 0; base < n; base += BPE_NT) {       // chunked so the scan carries across chunks
            int i = base + tid;
            int start = 0;
            if (i < n) {
                bool bd = symb[0][i] >= SYM_UNK;
                bool pb = (i > 0) && symb[0][i - 1] >= SYM_UNK;
                start = (i == 0 || bd || pb) ? 1 : 0;
            }
            int tot;
            int ex = bpe_exscan(start != 0, warp_tmp, pp, tot);
            uint32_t sg = 0, rk = BPE_INF;
            if (i < n) {
                sg = (uint32_t)(seg_base + ex + start - 1);
                segb[0][i] = (uint16_t)sg;
                if (start) { origin[sg] = (uint16_t)i; segstart[sg] = (uint16_t)i; }
                rk = (i + 1 < n) ? bpe_rank(A, symb[0][i], symb[0][i + 1]) : BPE_INF;
                rnkb[0][i] = (uint16_t)rk;
            }
            bpe_warp_seg_min(sminb[0], sg, rk, i < n);
            seg_base += tot;
        }
        __syncthreads();

        // ---- rounds ----------------------------------------------------------------------
        while (n > 0) {
            uint16_t *sym = symb[cur], *rnk = rnkb[cur], *seg = segb[cur], *segmin = sminb[ms];
            uint16_t *sym2 = symb[cur ^ 1], *rnk2 = rnkb[cur ^ 1], *seg2 = segb[cur ^ 1], *smin2 = sminb[ms ^ 1];
            // the other minima buffer gets ready for the rank pass of this round
            for (int i = tid; i <= seg_base; i += BPE_NT) smin2[i] = (uint16_t)BPE_INF;
            // flags, run parity, compaction
            int carry = 0;
            for (int base = 0; base < n; base += BPE_NT) {
                int i = base + tid;
                bool keep = false, merge = false;
                {
                    auto fires = [&](int j) -> bool {            // pair (j, j+1) is selected (before overlap rule)
                        uint32_t rk = rnk[j];
                        return rk != BPE_INF && rk == segmin[seg[j]];
                    };
                    auto merges = [&](int j) -> bool {           // left to right, non-overlapping (Q11)
                        if (!fires(j)) return false;
                        int c = 0;
                        while (j - 1 - c >= 0 && fires(j - 1 - c)) ++c;
                        return (c & 1) == 0;
                    };
                    // one look at the symbol's own pair; the run of selected pairs in front of it comes from the warp's
                    // ballot, and only a run that reaches the warp's first lane is followed back through shared memory
                    const int ln = tid & 31;
                    // a finished segment leaves: its tokens go to their place in the read
                    const uint32_t sgi = i < n ? (uint32_t)seg[i] : 0u;
                    const bool fin = i < n && segmin[sgi] == BPE_INF;
                    if (fin) A.tmp_tok[k0 + origin[sgi] + (i - (int)segstart[sgi])] = sym[i];
                    const uint32_t fb = __ballot_sync(0xffffffffu, fin);
                    if (ln == 0 && fb) atomicAdd(&s_cnt, __popc(fb));
                    const bool f = i < n && !fin && fires(i);
                    const uint32_t Fw = __ballot_sync(0xffffffffu, f);
                    int c = ln ? __clz(~(Fw << (32 - ln))) : 0;  // selected pairs directly in front, inside the warp
                    if (c > ln) c = ln;
                    if (f && c == ln) { int j = i - ln - 1; while (j >= 0 && fires(j)) { ++c; --j; } }
                    merge = f && (c & 1) == 0;
                    const bool pm = __shfl_up_sync(0xffffffffu, merge, 1);
                    if (i < n && !fin) keep = !(ln ? pm : (i > 0 && merges(i - 1)));
                }
                int tot;
                int w = carry + bpe_exscan(keep, warp_tmp, pp, tot);
                if (keep) {
                    sym2[w] = merge ? (uint16_t)(4u + rnk[i]) : sym[i];
                    seg2[w] = seg[i];
                    if (i == 0 || seg[i - 1] != seg[i]) segstart[seg[i]] = (uint16_t)w;   // first symbol of its segment
                    src[w] = (uint16_t)(merge ? 0xffffu : i);    // 0xffff: freshly merged token
                }
                carry += tot;
            }
            __syncthreads();
            const int n2 = carry;
            for (int base = 0; base < n2; base += BPE_NT) {
                const int w = base + tid;
                uint32_t rk = BPE_INF, sg = 0;
                if (w < n2) {
                    if (w + 1 < n2 && seg2[w] == seg2[w + 1]) {      // neighbours of different segments never pair
                        if (src[w] == 0xffffu || src[w + 1] == 0xffffu) rk = bpe_rank(A, sym2[w], sym2[w + 1]);
                        else rk = rnk[src[w]];
                    }
                    rnk2[w] = (uint16_t)rk;
                    sg = seg2[w];
                }
                bpe_warp_seg_min(smin2, sg, rk, w < n2);
            }
            n = n2; cur ^= 1; ms ^= 1;
            __syncthreads();
        }
        if (tid == 0) A.tok_cnt[r] = s_cnt;     // every token has been written by the pass that retired its segment
    }
}

// single-block exclusive scan of per-read token counts -> out_offsets (int64), total in the last entry
__global__ void __launch_bounds__(1024) scan_counts_kernel(const int32_t *cnt, int64_t n, int64_t *out_off) {
    __shared__ long long wsum[32];
    __shared__ long long s_carry;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (tid == 0) s_carry = 0;
    __syncthreads();
    for (int64_t base = 0; base < n; base += 1024) {
        int64_t i = base + tid;
        long long v = (i < n) ? cnt[i] : 0, inc = v;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) { long long t = __shfl_up_sync(0xffffffffu, inc, d); if (lane >= d) inc += t; }
        if (lane == 31) wsum[warp] = inc;
        __syncthreads();
        long long woff = 0, tot = 0;
        for (int w = 0; w < 32; ++w) { long long t = wsum[w]; if (w < warp) woff += t; tot += t; }
        long long carry = s_carry;
        if (i < n) out_off[i] = carry + woff + inc - v;
        __syncthreads();
        if (tid == 0) s_carry = carry + tot;
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
            if (s != SYM_HOLE && at < o_end) {               // (a read that did not fit the workspace has no tokens)
                const int32_t id = s == SYM_N ? n_id : (s == SYM_UNK ? unk_id : (int32_t)(base_id + s));
                if (at < ids_cap) ids[at] = (IdT)id; else status[0] = 1u;
            }
            o += __popc(vm);
        }
    }
}

}  // namespace dtk
