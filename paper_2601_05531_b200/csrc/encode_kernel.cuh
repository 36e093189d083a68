// encode_kernel.cuh -- single-pass classify + strip + {single-nt | k-mer} + CSR offsets.
//
// One persistent CTA claims flat 8 KiB byte tiles in order (atomic ticket), so every
// predecessor of a claimed tile is already running: the look-back below cannot deadlock.
// Per tile:
//   1. cp.async the tile into shared memory (16-byte coalesced, zero-fill past the end)
//   2. classify every byte through the 256-entry LUT held in shared memory
//      -> per-word bitmaps (skip / newline / '>' ) + class bytes
//   3. line-state scan (only with strip_headers): a 3-bit summary per tile, resolved by
//      looking back to the nearest tile that contains a newline or a record start
//   4. keep = ~skip & ~header & in-record; popc + block prefix scan -> compact class array
//   5. tile aggregate (kept counts, tokens of records closed inside, k-1 trailing classes)
//      published; decoupled look-back gives the inclusive prefix (out_offsets of the open
//      record, its kept-base count, its pending partial window)
//   6. tokens are pulled from the compact array window by window and stored coalesced;
//      out_offsets[r] is written by the tile that holds record r's first byte.
// Input bytes are read from HBM exactly once and ids written exactly once.
#pragma once
#include "common.cuh"

namespace dtk {

struct TileSmem {
    alignas(16) uint8_t raw[TB];                 // raw bytes, then class codes in place
    alignas(16) uint8_t cls[PEND_MAX + TB];      // compact kept classes (PEND_MAX carried slots in front)
    uint32_t skip[NT], nl[NT], gt[NT], rs[NT], hd[NT], keep[NT];
    int32_t scan[NT];                            // exclusive kept-base prefix per 32-byte word
    int32_t ev_k[NT], ev_n[NT];                  // per-event kept prefix / kept count (one chunk of events)
    long long ev_out[NT];
    int32_t warp_tmp[NT / 32];
    uint8_t lut[256];
    int32_t tile, max_reset, ktot, blk_total;
    long long r_lo, r_hi;
    uint32_t ls_in;
    Prefix pin;
};

__device__ __forceinline__ void cp_async16(void *smem, const void *gmem, int src_bytes) {
    uint32_t s = (uint32_t)__cvta_generic_to_shared(smem);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(s), "l"(gmem), "r"(src_bytes) : "memory");
}
__device__ __forceinline__ void cp_async_wait_all() {
    asm volatile("cp.async.commit_group;\ncp.async.wait_group 0;" ::: "memory");
}

// exclusive block scan of one int per thread; total broadcast through sm.blk_total
__device__ __forceinline__ int block_exscan(int v, TileSmem &sm, int &total) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    int inc = v;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) { int t = __shfl_up_sync(0xffffffffu, inc, d); if (lane >= d) inc += t; }
    if (lane == 31) sm.warp_tmp[warp] = inc;
    __syncthreads();
    int woff = 0, tot = 0;
#pragma unroll
    for (int w = 0; w < NT / 32; ++w) { int t = sm.warp_tmp[w]; if (w < warp) woff += t; tot += t; }
    __syncthreads();
    total = tot;
    return woff + inc - v;
}

// position of record offset index r, relative to nothing (absolute "position" space)
__device__ __forceinline__ int64_t rec_pos(const EncArgs &A, int64_t r) { return A.rec_off[r] - A.off_bias + A.mis; }

// first r in [lo, n_rec + 1) with rec_pos(r) >= pos; warp-cooperative 32-ary search (all lanes return it)
__device__ __forceinline__ int64_t warp_lower_bound(const EncArgs &A, int64_t lo, int64_t pos) {
    const int lane = threadIdx.x & 31;
    int64_t hi = A.n_rec + 1;                    // answer in [lo, hi]
    while (hi - lo > 32) {
        int64_t step = (hi - lo + 31) / 32;      // probe lo + (lane+1)*step - 1
        int64_t idx = lo + (int64_t)(lane + 1) * step - 1;
        bool ge = (idx >= hi) ? true : (rec_pos(A, idx) >= pos);
        uint32_t b = __ballot_sync(0xffffffffu, ge);
        if (!b) return hi;                       // lane 31 probed hi-1 and even that is < pos
        int f = __ffs(b) - 1;                    // first probe that is >= pos (lane 31 probes >= hi-1 or beyond)
        int64_t nlo = lo + (int64_t)f * step;    // everything before probe f-1 (inclusive) is < pos
        int64_t nhi = lo + (int64_t)(f + 1) * step - 1;
        if (nhi > hi) nhi = hi;
        lo = nlo; hi = nhi;
    }
    int64_t idx = lo + lane;
    bool ge = (idx >= hi) ? true : (rec_pos(A, idx) >= pos);
    uint32_t b = __ballot_sync(0xffffffffu, ge);
    return b ? lo + (__ffs(b) - 1) : hi;         // hi - lo == 32: no lane probed hi itself
}

__device__ __forceinline__ int kept_before(const TileSmem &sm, int p) {   // kept bases at tile positions < p
    if (p >= TB) return sm.ktot;
    return sm.scan[p >> 5] + __popc(sm.keep[p >> 5] & ((1u << (p & 31)) - 1u));
}

__device__ __forceinline__ int next_reset(const TileSmem &sm, int from) {  // first nl|rs bit at >= from, else TB
    if (from >= TB) return TB;
    int w = from >> 5;
    uint32_t m = (sm.nl[w] | sm.rs[w]) & (~0u << (from & 31));
    while (!m && ++w < NT) m = sm.nl[w] | sm.rs[w];
    return m ? w * 32 + __ffs(m) - 1 : TB;
}

__device__ __forceinline__ void mark_range(TileSmem &sm, int a, int b) {   // set hd bits [a, b]
    for (int w = a >> 5; w <= (b >> 5); ++w) {
        uint32_t m = ~0u;
        if (w == (a >> 5)) m &= ~0u << (a & 31);
        if (w == (b >> 5)) m &= ~0u >> (31 - (b & 31));
        atomicOr(&sm.hd[w], m);
    }
}

// first byte at >= s that is not a non-newline SKIP byte (those leave line_start unchanged, Q3); TB if none
__device__ __forceinline__ int skip_other_skips(const TileSmem &sm, int s) {
    while (s < TB && (((sm.skip[s >> 5] & ~sm.nl[s >> 5]) >> (s & 31)) & 1u)) ++s;
    return s;
}

// a line starts at tile position s: if its first byte is '>' drop it through the next '\n' (inclusive) or
// up to the next record start (exclusive) or the tile's end (Q4)
__device__ __forceinline__ void mark_header_from(TileSmem &sm, int s) {
    s = skip_other_skips(sm, s);
    if (s >= TB || !((sm.gt[s >> 5] >> (s & 31)) & 1u)) return;
    int e = next_reset(sm, s + 1);
    if (e >= TB) e = TB - 1;
    else if ((sm.rs[e >> 5] >> (e & 31)) & 1u) e -= 1;
    mark_range(sm, s, e);
}

template <typename IdT>
__device__ __forceinline__ void store_id(const EncArgs &A, int64_t idx, int32_t id) {
    if (idx < A.ids_cap) reinterpret_cast<IdT *>(A.ids)[idx] = (IdT)id;
    else A.status[0] = 1u;
}

// emit the tokens of one record piece from the compact class array.
//   src: index into sm.cls of its first not-yet-consumed kept base; n: kept bases available;
//   closes: the record ends inside this tile (emit the tail); g/gs: index within / size of the thread group
template <typename IdT>
__device__ __forceinline__ void emit_segment(const EncArgs &A, const TileSmem &sm, int src, int n, bool closes,
                                             int64_t out_base, int g, int gs) {
    const EncParams &P = A.prm;
    if (P.mode == MODE_KMER) {
        const int k = P.k, nwin = n / k, rem = n - nwin * k;
        for (int w = g; w < nwin; w += gs) {
            const uint8_t *c = sm.cls + src + w * k;
            uint32_t code = 0, bad = 0;
            for (int i = 0; i < k; ++i) { uint32_t ci = c[i]; bad |= ci; code = code * 4u + (ci & 3u); }
            store_id<IdT>(A, out_base + w, (bad & 4u) ? P.unk_id : (int32_t)(P.base_id + code));
        }
        if (closes && rem) {
            if (P.tail_policy == TAIL_PER_BASE) {
                for (int i = g; i < rem; i += gs) {
                    uint32_t ci = sm.cls[src + nwin * k + i];
                    store_id<IdT>(A, out_base + nwin + i, ci <= CLS_N ? (int32_t)(P.base_id + P.four_k + ci) : P.unk_id);
                }
            } else if (P.tail_policy == TAIL_UNK) {
                if (g == 0) store_id<IdT>(A, out_base + nwin, P.unk_id);
            }
        }
    } else {
        for (int i = g; i < n; i += gs) {
            uint32_t ci = sm.cls[src + i];
            store_id<IdT>(A, out_base + i, ci <= CLS_N ? P.nt_ids[ci] : P.unk_id);
        }
    }
}

template <typename IdT>
__global__ void __launch_bounds__(NT) encode_tiles_kernel(const __grid_constant__ EncArgs A) {
    extern __shared__ __align__(16) uint8_t smem_raw[];
    TileSmem &sm = *reinterpret_cast<TileSmem *>(smem_raw);
    const EncParams &P = A.prm;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const uint32_t gen = A.gen;

    sm.lut[tid] = A.lut[tid];
    const int64_t pos_first = rec_pos(A, 0), pos_last = rec_pos(A, A.n_rec);   // bytes outside are in no record

    for (;;) {
        __syncthreads();
        if (tid == 0) sm.tile = (int)(atomicAdd(A.ticket, 1ull) - A.ticket_base);
        __syncthreads();
        const int tile = sm.tile;
        if (tile >= A.n_tiles) break;
        const int64_t t0 = (int64_t)tile * TB;
        TileDesc &D = A.descs[tile];

        // ---- 1. load ------------------------------------------------------------------
#pragma unroll
        for (int i = 0; i < TB / NT / 16; ++i) {
            int c = tid + i * NT;
            int64_t p = t0 + (int64_t)c * 16;
            cp_async16(sm.raw + c * 16, A.bytes_al + (p < A.p_end ? p : 0), p < A.p_end ? 16 : 0);
        }
        // ---- events of this tile (record offsets that fall inside it), while the copy is in flight
        if (warp == 0) {
            int64_t rlo = warp_lower_bound(A, 0, t0);
            int64_t rhi = (tile == A.n_tiles - 1) ? A.n_rec + 1 : warp_lower_bound(A, rlo, t0 + TB);
            if (lane == 0) { sm.r_lo = rlo; sm.r_hi = rhi; sm.max_reset = -1; }
        }
        sm.rs[tid] = 0; sm.hd[tid] = 0;
        cp_async_wait_all();
        __syncthreads();
        const int64_t r_lo = sm.r_lo;
        const int m = (int)(sm.r_hi - r_lo);                 // events in this tile

        // ---- 2. classify my 32 bytes ---------------------------------------------------
        uint32_t skip = 0, nl = 0, gt = 0;
        {
            uint32_t *w = reinterpret_cast<uint32_t *>(sm.raw + tid * SPAN);
#pragma unroll
            for (int q = 0; q < SPAN / 4; ++q) {
                uint32_t x = w[q], y = 0;
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    uint32_t b = (x >> (8 * j)) & 0xffu, c = sm.lut[b];
                    y |= c << (8 * j);
                    skip |= (uint32_t)(c == CLS_SKIP) << (q * 4 + j);
                    nl |= (uint32_t)(b == '\n') << (q * 4 + j);
                    gt |= (uint32_t)(b == '>') << (q * 4 + j);
                }
                w[q] = y;
            }
            sm.skip[tid] = skip; sm.nl[tid] = nl; sm.gt[tid] = gt;
        }
        for (int e = tid; e < m; e += NT) {
            int p = (int)(rec_pos(A, r_lo + e) - t0);
            atomicOr(&sm.rs[p >> 5], 1u << (p & 31));
        }
        __syncthreads();

        // ---- 3. line state + header lines ----------------------------------------------
        if (P.strip_headers) {
            int cand = -1;                                   // last line start inside the tile
            if (nl) cand = tid * 32 + (31 - __clz(nl)) + 1;
            uint32_t rs = sm.rs[tid];
            if (rs) cand = max(cand, tid * 32 + (31 - __clz(rs)));
            cand = __reduce_max_sync(0xffffffffu, cand);
            if (lane == 0 && cand >= 0) atomicMax(&sm.max_reset, cand);
            __syncthreads();
            if (tid == 0) {
                const bool has_reset = sm.max_reset >= 0;
                int s = skip_other_skips(sm, has_reset ? sm.max_reset : 0);
                uint32_t x = (s >= TB) ? LS_LINE_START : (((sm.gt[s >> 5] >> (s & 31)) & 1u) ? LS_IN_HEADER : LS_IN_LINE);
                st_release(&D.l_word, (gen << 8) | ((uint32_t)has_reset << 2) | x);
                // entry state: walk back to the nearest tile whose exit state is known
                uint32_t g_s = LS_LINE_START, ls_in = LS_LINE_START;
                bool ok = true;
                for (int j = tile - 1; j >= 0; --j) {
                    const TileDesc &Dj = A.descs[j];
                    uint32_t v = 0; bool done = false; int spins = 0;
                    for (;;) {
                        v = ld_acquire(&Dj.l_incl);
                        if ((v >> 8) == gen) { v &= 3u; done = true; break; }
                        v = ld_acquire(&Dj.l_word);
                        if ((v >> 8) == gen) { done = (v >> 2) & 1u; v &= 3u; break; }
                        if (++spins > SPIN_LIMIT) { ok = false; break; }
                    }
                    if (!ok) break;
                    if (done || j == 0) { ls_in = (v == LS_LINE_START) ? g_s : v; break; }
                    if (v != LS_LINE_START) g_s = v;         // prepend f_j: g(S) := g(x_j)
                }
                if (!ok) A.status[1] = 1u;
                sm.ls_in = ls_in;
                uint32_t ex = has_reset ? x : (ls_in == LS_LINE_START ? x : ls_in);
                st_release(&D.l_incl, (gen << 8) | ex);
            }
            // header lines that start inside the tile: after each '\n', at each record start
            for (uint32_t b = nl; b; b &= b - 1) mark_header_from(sm, tid * 32 + __ffs(b));
            for (int e = tid; e < m; e += NT) mark_header_from(sm, (int)(rec_pos(A, r_lo + e) - t0));
            __syncthreads();
            if (tid == 0) {                                  // the line that straddles the tile's start
                if (sm.ls_in == LS_IN_HEADER) {
                    int e = next_reset(sm, 0);
                    if (e >= TB) e = TB - 1;
                    else if ((sm.rs[e >> 5] >> (e & 31)) & 1u) e -= 1;
                    if (e >= 0) mark_range(sm, 0, e);
                } else if (sm.ls_in == LS_LINE_START) {
                    mark_header_from(sm, 0);
                }
            }
            __syncthreads();
        }

        // ---- 4. keep mask, prefix scan, compaction --------------------------------------
        uint32_t keep = ~skip & ~sm.hd[tid];
        {
            int64_t a = pos_first - t0 - (int64_t)tid * 32, b = pos_last - t0 - (int64_t)tid * 32;
            uint32_t ma = a <= 0 ? ~0u : (a >= 32 ? 0u : (~0u << a));
            uint32_t mb = b <= 0 ? 0u : (b >= 32 ? ~0u : ((1u << b) - 1u));
            keep &= ma & mb;
        }
        sm.keep[tid] = keep;
        int ktot;
        int pos = block_exscan(__popc(keep), sm, ktot);
        sm.scan[tid] = pos;
        if (tid == 0) sm.ktot = ktot;
        {
            const uint8_t *c = sm.raw + tid * SPAN;
            uint8_t *o = sm.cls + PEND_MAX + pos;
#pragma unroll
            for (int j = 0; j < SPAN; ++j)
                if ((keep >> j) & 1u) *o++ = c[j];
        }
        __syncthreads();

        // ---- 5. aggregate, look-back, inclusive prefix ----------------------------------
        int first_kept = ktot, last_kept = ktot;
        int closed_part = 0;
        if (m > 0) {
            first_kept = kept_before(sm, (int)(rec_pos(A, r_lo) - t0));
            last_kept = ktot - kept_before(sm, (int)(rec_pos(A, r_lo + m - 1) - t0));
            for (int e = tid; e < m - 1; e += NT) {
                int ka = kept_before(sm, (int)(rec_pos(A, r_lo + e) - t0));
                int kb = kept_before(sm, (int)(rec_pos(A, r_lo + e + 1) - t0));
                closed_part += (int)tok_count(kb - ka, P);
            }
        }
        int closed_tokens;
        (void)block_exscan(closed_part, sm, closed_tokens);
        if (tid == 0) {
            Agg G;
            G.first_kept = first_kept; G.last_kept = last_kept; G.closed_tokens = closed_tokens; G.has_event = m > 0;
            uint32_t tn = (uint32_t)min(P.k - 1, last_kept);
            uint64_t tl = 0;
            for (uint32_t i = 0; i < tn; ++i) tl = (tl << 4) | sm.cls[PEND_MAX + ktot - (int)tn + (int)i];
            G.tail = tl; G.tail_cnt = tn;
            Prefix X; X.T = 0; X.open_n = 0; X.tail = 0; X.tail_cnt = 0;
            if (tile > 0) {
                D.has_event = G.has_event; D.first_kept = first_kept; D.last_kept = last_kept;
                D.closed_tokens = closed_tokens; D.tail = tl; D.tail_cnt = tn;
                st_release(&D.status, (gen << 2) | ST_AGG);
                Agg acc; bool have = false, ok = true;
                for (int j = tile - 1; j >= 0; --j) {
                    const TileDesc &Dj = A.descs[j];
                    uint32_t st; int spins = 0;
                    while ((((st = ld_acquire(&Dj.status)) >> 2) != gen || (st & 3u) == ST_EMPTY)) {
                        if (++spins > SPIN_LIMIT) { ok = false; break; }
                    }
                    if (!ok) break;
                    if ((st & 3u) == ST_INCL) {
                        X.T = Dj.T; X.open_n = Dj.open_n; X.tail = Dj.ptail; X.tail_cnt = Dj.ptail_cnt;
                        break;
                    }
                    Agg Aj;
                    Aj.first_kept = Dj.first_kept; Aj.last_kept = Dj.last_kept; Aj.closed_tokens = Dj.closed_tokens;
                    Aj.tail = Dj.tail; Aj.tail_cnt = Dj.tail_cnt; Aj.has_event = Dj.has_event;
                    acc = have ? agg_compose(Aj, acc, P) : Aj;
                    have = true;
                }
                if (!ok) A.status[1] = 1u;
                if (have) X = prefix_apply(X, acc, P);
            }
            sm.pin = X;
            Prefix Y = prefix_apply(X, G, P);
            D.T = Y.T; D.open_n = Y.open_n; D.ptail = Y.tail; D.ptail_cnt = Y.tail_cnt;
            st_release(&D.status, (gen << 2) | ST_INCL);
            // carried bases of the open record go in front of the compact array
            int pend = (P.mode == MODE_KMER) ? (int)(X.open_n % P.k) : 0;
            for (int i = 0; i < pend; ++i) sm.cls[PEND_MAX - pend + i] = (uint8_t)((X.tail >> (4 * (pend - 1 - i))) & 0xfu);
        }
        __syncthreads();

        // ---- 6. emit ---------------------------------------------------------------------
        const Prefix X = sm.pin;
        const int pend = (P.mode == MODE_KMER) ? (int)(X.open_n % P.k) : 0;
        {   // the record that was open at the tile's start
            int64_t done = (P.mode == MODE_KMER) ? X.open_n / P.k : X.open_n;
            emit_segment<IdT>(A, sm, PEND_MAX - pend, pend + first_kept, m > 0, A.out_bias + X.T + done, tid, NT);
        }
        if (m > 0) {
            int64_t base_T = A.out_bias + X.T + tok_count(X.open_n + first_kept, P);   // = out_offsets[r_lo]
            for (int c0 = 0; c0 < m; c0 += NT) {
                const int e = c0 + tid, cm = min(NT, m - c0);
                int ke = 0, ne = 0, te = 0;
                if (e < m) {
                    ke = kept_before(sm, (int)(rec_pos(A, r_lo + e) - t0));
                    int kn = (e + 1 < m) ? kept_before(sm, (int)(rec_pos(A, r_lo + e + 1) - t0)) : ktot;
                    ne = kn - ke;
                    te = (e + 1 < m) ? (int)tok_count(ne, P) : 0;
                }
                int chunk_total;
                int ex = block_exscan(te, sm, chunk_total);
                if (e < m) {
                    A.out_off[r_lo + e] = base_T + ex;
                    sm.ev_k[tid] = ke; sm.ev_n[tid] = ne; sm.ev_out[tid] = base_T + ex;
                }
                __syncthreads();
                if (cm <= 8) {
                    for (int i = 0; i < cm; ++i)
                        if (r_lo + c0 + i < A.n_rec)
                            emit_segment<IdT>(A, sm, PEND_MAX + sm.ev_k[i], sm.ev_n[i], c0 + i + 1 < m, sm.ev_out[i], tid, NT);
                } else {
                    for (int i = warp; i < cm; i += NT / 32)
                        if (r_lo + c0 + i < A.n_rec)
                            emit_segment<IdT>(A, sm, PEND_MAX + sm.ev_k[i], sm.ev_n[i], c0 + i + 1 < m, sm.ev_out[i], lane, 32);
                }
                base_T += chunk_total;
                __syncthreads();
            }
        }
    }
}

}  // namespace dtk
