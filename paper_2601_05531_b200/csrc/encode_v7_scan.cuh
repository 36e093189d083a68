// encode_v7_scan.cuh -- the scan warp's jobs: tile preparation, aggregate + publication, line-state check, prefix
// (look-back, or closed form in DENSE mode), segment table, out_offsets, halo.  Included by encode_v7.cuh.
#pragma once

namespace dtk {
namespace v7 {

// ---- preparation of a tile: record range, record-start list, L2 prefetch ------------------------------------------
__device__ __forceinline__ int scan_prep(const EncArgs &A, TileBuf &tb, unsigned long long ticket, int lane) {
    const unsigned long long rel = ticket - A.ticket_base;
    if (rel >= (unsigned long long)A.n_tiles) return -1;
    const int tile = (int)rel;
    const int64_t TBS = (int64_t)A.S * TB;
    const int64_t t0 = (int64_t)tile * TBS;
    if (lane < A.S) prefetch_l2(A, t0 + (int64_t)lane * TB, TB);
    const int64_t rlo = A.first_rec[tile], rhi = A.first_rec[tile + 1];
    const int64_t m64 = rhi - rlo;
    const int m = m64 > 0x7fffffff ? 0x7fffffff : (int)m64;
    if (m <= EV_MAX)
        for (int e = lane; e < m; e += 32) tb.ev_p[e] = (uint16_t)(rec_pos(A, rlo + e) - t0);
    if (lane == 0) { tb.tile = tile; tb.m = m; tb.rlo = rlo; }
    __syncwarp();
    return tile;
}

// ---- entry line state of a tile from the chain of per-tile words (tile > 0) -----------------------------------------
__device__ __noinline__ uint32_t ls_chain_state(const EncArgs &A, int tile, int lane) {
    constexpr uint32_t FULL = 0xffffffffu;
    const uint32_t gen = A.gen;
    bool ok = true;
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
            __nanosleep(40);
        }
        if (!ok) break;
        // the value that survives is the farthest non-LINE_START one at or before the final tile
        const uint32_t nb = __ballot_sync(FULL, val != LS_LINE_START && lane <= f);
        if (nb) { carry = __shfl_sync(FULL, val, 31 - __clz(nb)); have_carry = true; }
        if (f < 32) break;
    }
    if (!ok && lane == 0) A.status[1] = 1u;
    return have_carry ? carry : LS_LINE_START;
}

// ---- after the compute warps finished a tile: line-state check, region prefix ---------------------------------------
// A region that assumed IN_LINE but really started inside a header line loses the kept bases in front of its first
// line reset: its first slot moves up by that many (rbase) and its count shrinks.
template <bool DENSE>
__device__ __forceinline__ void scan_regions(const EncArgs &A, TileBuf &tb, int lane) {
    constexpr uint32_t FULL = 0xffffffffu;
    const EncParams &P = A.prm;
    const int tile = tb.tile;
    const int64_t TBS = (int64_t)A.S * TB, t0 = (int64_t)tile * TBS;
    if (DENSE) {
        const int RB = A.S * WB;
        if (lane <= NWC) tb.cum[lane] = lane * RB;
        if (lane < NWC) tb.rbase[lane] = reg_slot(lane);
        if (lane == 0) {
            const int64_t rem = rec_pos(A, A.n_rec) - t0;
            tb.ktot = rem < 0 ? 0 : (rem > TBS ? (int)TBS : (int)rem);
        }
        __syncwarp();
        return;
    }
    uint32_t dropmask = 0;                                 // regions that started inside a header line unawares
    if (P.strip_headers) {
        const uint32_t tagL = A.gen << 8;
        uint32_t rl[NWC];
#pragma unroll
        for (int w = 0; w < NWC; ++w) rl[w] = tb.reg_ls[w];
        uint32_t t_hr = 0, t_x = LS_LINE_START;            // summary of the whole tile
#pragma unroll
        for (int w = 0; w < NWC; ++w) { t_x = ls_apply((rl[w] >> 2) & 1u, rl[w] & 3u, t_x); t_hr |= (rl[w] >> 2) & 1u; }
        uint32_t state = (rl[0] >> 4) & 3u;                // entry state of the tile
        if (!((rl[0] >> 8) & 1u)) {
            // region 0 ran under an assumption: publish what is known, then ask the chain
            if (lane == 0) st_vol32(&A.ls[tile], tagL | ((t_hr ? LK_FINAL : LK_SUMMARY) << 2) | t_x);
            state = ls_chain_state(A, tile, lane);
        }
        if (lane == 0) st_vol32(&A.ls[tile], tagL | (LK_FINAL << 2) | ls_apply(t_hr, t_x, state));
#pragma unroll
        for (int w = 0; w < NWC; ++w) {
            if (!((rl[w] >> 8) & 1u) && state == LS_IN_HEADER) dropmask |= 1u << w;
            state = ls_apply((rl[w] >> 2) & 1u, rl[w] & 3u, state);
        }
    }
    const int drop = (lane < NWC && ((dropmask >> lane) & 1u)) ? tb.reg_hfix[lane] : 0;
    int c = lane < NWC ? tb.reg_cnt[lane] - drop : 0, inc = c;
#pragma unroll
    for (int d = 1; d < NWC; d <<= 1) { const int t = __shfl_up_sync(FULL, inc, d); if (lane >= d) inc += t; }
    if (lane < NWC) { tb.cum[lane] = inc - c; tb.rbase[lane] = reg_slot(lane) + drop; }
    if (lane == NWC - 1) { tb.cum[NWC] = inc; tb.ktot = inc; }
    __syncwarp();
}

// logical kept-base index in front of record start e of the tile
template <bool DENSE>
__device__ __forceinline__ int event_kept(const EncArgs &A, const TileBuf &tb, int e, int64_t t0) {
    if (tb.m <= EV_MAX) return DENSE ? (int)tb.ev_p[e] : tb.ev_k[e];
    return DENSE ? (int)(rec_pos(A, tb.rlo + e) - t0) : __ldcg(A.rec_k + tb.rlo + e);
}

// ---- aggregate of a tile and its logical entries (one per record start) -------------------------------------------
// le_t holds token indices relative to the first record start (entry 0's tokens are added once the prefix is known).
template <bool DENSE>
__device__ __forceinline__ void scan_aggregate(const EncArgs &A, TileBuf &tb, const uint32_t *st, int lane) {
    constexpr uint32_t FULL = 0xffffffffu;
    const EncParams &P = A.prm;
    const int k = P.k, m = tb.m, ktot = tb.ktot, tile = tb.tile;
    const int64_t t0 = (int64_t)tile * A.S * TB;
    if (!DENSE) {
        // region-relative -> logical
        if (m <= EV_MAX) {
            for (int e = lane; e < m; e += 32) {
                const int v = tb.ev_k[e], w = v >> 16;
                tb.ev_k[e] = max((v & 0xffff) - (tb.rbase[w] - reg_slot(w)), 0) + tb.cum[w];
            }
        } else {
            for (int e = lane; e < m; e += 32) {
                const int v = __ldcg(A.rec_k + tb.rlo + e), w = v >> 16;
                A.rec_k[tb.rlo + e] = max((v & 0xffff) - (tb.rbase[w] - reg_slot(w)), 0) + tb.cum[w];
            }
        }
        __syncwarp();
    }
    int fk = ktot, lk = ktot, closed = 0, ntok_ev = 0;
    if (m > 0) {
        int carry = 0;
        for (int c0 = 0; c0 < m; c0 += 32) {
            const int e = c0 + lane;
            const int ke = e < m ? event_kept<DENSE>(A, tb, e, t0) : ktot;
            int kn = __shfl_down_sync(FULL, ke, 1);
            if (lane == 31) kn = e + 1 < m ? event_kept<DENSE>(A, tb, e + 1, t0) : ktot;
            if (e >= m - 1) kn = ktot;
            const int ne = e < m ? kn - ke : 0;
            const int nw = (int)div_k((uint32_t)ne, P);
            // records that close inside emit windows + tail; the one still open at the end only windows
            const int te = e < m - 1 ? nw + tail_tokens(ne - nw * k, P) : (e == m - 1 ? nw : 0);
            int ti = te;
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) { const int t = __shfl_up_sync(FULL, ti, d); if (lane >= d) ti += t; }
            const int ex = carry + ti - te;
            if (m <= EV_MAX && e < m) { tb.le_src[1 + e] = ke; tb.le_t[1 + e] = ex; tb.le_nwin[1 + e] = nw; }
            if (c0 == 0) fk = __shfl_sync(FULL, ke, 0);
            if (c0 + 32 >= m) { lk = __shfl_sync(FULL, ne, m - 1 - c0); closed = __shfl_sync(FULL, ex, m - 1 - c0); }
            carry += __shfl_sync(FULL, ti, 31);
        }
        ntok_ev = carry;
    }
    // last tn = min(k - 1, lk) classes of the tile, 3 bits each, newest lowest
    const int tn = min(k - 1, lk);
    unsigned long long gtail = 0;
    if (!DENSE) {
        unsigned long long tl = 0;
        if (lane < tn) tl = (unsigned long long)class_at(st, slot_of(tb, ktot - tn + lane)) << (3 * (tn - 1 - lane));
        gtail = ((unsigned long long)__reduce_or_sync(FULL, (uint32_t)(tl >> 32)) << 32) | __reduce_or_sync(FULL, (uint32_t)tl);
    }
    if (lane == 0) {
        if (!DENSE) {
            const uint32_t tagA = (A.gen << 2) | ST_AGG;
            TileDesc &D = A.descs[tile];
            st_vol128(&D.a0, make_uint4(tagA, (uint32_t)fk, (uint32_t)lk, (uint32_t)closed | ((uint32_t)(m > 0) << 31)));
            st_vol128(&D.a1, make_uint4(tagA, (uint32_t)tn | ((uint32_t)(gtail >> 32) << 4), (uint32_t)gtail, 0u));
        }
        TileAgg &g = tb.ag;
        g.fk = fk; g.lk = lk; g.closed = closed; g.tn = tn; g.hasev = m > 0; g.tail = gtail;
        tb.ntok = ntok_ev;
        tb.e_tile = tile; tb.e_m = m; tb.e_rlo = tb.rlo;   // (tile / m / rlo / ev_p belong to the next tile's preparation from here on)
    }
    __syncwarp();
}

// class c (0..5) into stream slot u, whatever the slot held (single lanes of the scan warp; other lanes may hit the same word)
__device__ __forceinline__ void put_class(uint32_t *st, int u, uint32_t c) {
    const uint32_t dg = c < CLS_N ? c : (c == CLS_N ? 2u : 1u);
    const int sh = 30 - 2 * (u & 15);
    atomicAnd(&st[u >> 4], ~(3u << sh));
    atomicOr(&st[u >> 4], dg << sh);
    const uint32_t fb = 1u << (31 - (u & 31));
    if (c >= CLS_N) atomicOr(&st[SW_CODE + (u >> 5)], fb); else atomicAnd(&st[SW_CODE + (u >> 5)], ~fb);
}

// ---- prefix of a tile, its segment table, out_offsets, halo -------------------------------------------------------
// Returns false (nothing changed) when a predecessor the look-back needs has not published yet.
template <bool DENSE>
__device__ __forceinline__ bool scan_tables(const EncArgs &A, const Smem7 &sm, TileBuf &tb, uint32_t *st, int lane, bool force) {
    constexpr uint32_t FULL = 0xffffffffu;
    const EncParams &P = A.prm;
    const int k = P.k, m = tb.e_m, tile = tb.e_tile, ktot = tb.ktot;
    const int64_t t0 = (int64_t)tile * A.S * TB, rlo = tb.e_rlo;
    auto kept = [&](int e) -> int { return DENSE ? (int)(rec_pos(A, rlo + e) - t0) : __ldcg(A.rec_k + rlo + e); };   // (m > EV_MAX only)
    const TileAgg g = tb.ag;
    int pend, nwin0, tok0;
    int64_t T0;
    if (!DENSE) {
        bool ready;
        Agg ga; ga.hasev = g.hasev; ga.fk = g.fk; ga.lk = g.lk; ga.closed = g.closed; ga.tn = g.tn; ga.tail = g.tail;
        const Pre X = look_back(A, tile, ga, lane, force, ready);
        if (!ready) return false;
        pend = P.mode == MODE_KMER ? X.o.r : 0;
        const int nbase0 = pend + g.fk;
        nwin0 = (int)div_k((uint32_t)nbase0, P);
        tok0 = nwin0 + (g.hasev ? tail_tokens(nbase0 - nwin0 * k, P) : 0);
        const Pre Y = pre_extend(X, ga, P);
        if (lane == 0) {
            const uint32_t tagI = (A.gen << 2) | ST_INCL;
            TileDesc &D = A.descs[tile];
            st_vol128(&D.i0, make_uint4(tagI, (uint32_t)Y.T, (uint32_t)((uint64_t)Y.T >> 32),
                                        (uint32_t)Y.o.r | ((uint32_t)Y.cnt << 4) | ((uint32_t)(Y.tail >> 32) << 8)));
            st_vol128(&D.i1, make_uint4(tagI, (uint32_t)Y.o.q, (uint32_t)((uint64_t)Y.o.q >> 32), (uint32_t)Y.tail));
        }
        // carried bases of the open record go right in front of region 0's first kept base
        if (lane < pend) put_class(st, tb.rbase[0] - pend + lane, (uint32_t)(X.tail >> (3 * (pend - 1 - lane))) & 7u);
        T0 = A.out_bias + X.T + X.o.q;
    } else {
        // closed form: the open record started at a known byte, every byte before the tile is a kept base
        pend = 0; nwin0 = 0; tok0 = 0;
        T0 = rlo <= A.n_rec ? __ldg(A.out_off + (rlo > 0 ? rlo - 1 : 0)) : 0;
        if (rlo > 0) {
            const int64_t nb = t0 - rec_pos(A, rlo - 1);
            const int64_t q = nb / k;
            pend = P.mode == MODE_KMER ? (int)(nb - q * k) : 0;
            T0 += P.mode == MODE_KMER ? q : nb;
            const int nbase0 = pend + g.fk;
            nwin0 = (int)div_k((uint32_t)nbase0, P);
            tok0 = nwin0 + (g.hasev ? tail_tokens(nbase0 - nwin0 * k, P) : 0);
            if (lane < pend) put_class(st, tb.rbase[0] - pend + lane, sm.lut[__ldg(A.bytes_al + t0 - pend + lane)]);
        }
    }
    const int ntok = tb.ntok + tok0;
    if (lane == 0) { tb.T0 = T0; tb.ntok = ntok; tb.pend = pend; tb.tok0 = tok0; tb.nwin0 = nwin0; }
    __syncwarp();
    if (m > EV_MAX) {
        // per-token fallback emission: only out_offsets are prepared here (records that start inside the tile)
        if (!DENSE) {
            long long carry = T0 + tok0;
            for (int c0 = 0; c0 < m; c0 += 32) {
                const int e = c0 + lane;
                const int ke = e < m ? kept(e) : ktot;
                int kn = __shfl_down_sync(FULL, ke, 1);
                if (lane == 31) kn = e + 1 < m ? kept(e + 1) : ktot;
                if (e >= m - 1) kn = ktot;
                const int ne = e < m ? kn - ke : 0;
                const int nw = (int)div_k((uint32_t)ne, P);
                const int te = e < m - 1 ? nw + tail_tokens(ne - nw * k, P) : (e == m - 1 ? nw : 0);
                int ti = te;
#pragma unroll
                for (int d = 1; d < 32; d <<= 1) { const int t = __shfl_up_sync(FULL, ti, d); if (lane >= d) ti += t; }
                if (e < m) A.out_off[rlo + e] = carry + ti - te;
                carry += __shfl_sync(FULL, ti, 31);
            }
            __threadfence();
        }
    } else {
        // ---- logical entries get entry 0's tokens; out_offsets of the records that start here --------------------
        for (int e = lane; e < m; e += 32) {
            const int t = tb.le_t[1 + e] + tok0;
            tb.le_t[1 + e] = t;
            if (!DENSE) A.out_off[rlo + e] = T0 + t;
        }
        if (lane == 0) { tb.le_src[0] = -pend; tb.le_t[0] = 0; tb.le_nwin[0] = nwin0; tb.le_t[m + 1] = ntok; }
        __syncwarp();
        // ---- split at the region starts: entry j >= 1 keeps its order behind the region starts at or before it ---
        for (int j0 = 1; j0 <= m; j0 += 32) {
            const int j = j0 + lane;
            if (j <= m) {
                const int ls = tb.le_src[j];
                int reg = 0;
#pragma unroll
                for (int w = 1; w < NWC; ++w) reg += (tb.cum[w] <= ls) ? 1 : 0;
                const int rank = j + reg;
                tb.se_src[rank] = tb.rbase[reg] + (ls - tb.cum[reg]);
                tb.se_t[rank] = tb.le_t[j];
                tb.se_nwin[rank] = tb.le_nwin[j];
            }
        }
        if (lane == 0) {
            tb.se_src[0] = tb.rbase[0] - pend; tb.se_t[0] = 0; tb.se_nwin[0] = nwin0;
            tb.reg_e0[0] = 0; tb.reg_e0[NWC] = m + NWC; tb.se_t[m + NWC] = ntok;
        } else if (lane < NWC) {
            const int c = tb.cum[lane];
            int lo = 0, hi = m;                            // record starts in front of the region start
            while (lo < hi) {
                const int mid = (lo + hi) >> 1;
                if (tb.le_src[1 + mid] < c) lo = mid + 1; else hi = mid;
            }
            const int j = lo;                              // the entry the region start falls into
            const int src = tb.le_src[j], tj = tb.le_t[j], nwj = tb.le_nwin[j], nt = tb.le_t[j + 1] - tj - nwj;
            const int d = c - src;
            const int jw = min(nwj, (d + k - 1) / k);      // windows whose first base lies in front of the region
            int ls, t, nw;
            if (jw < nwj) { ls = src + jw * k; t = tj + jw; nw = nwj - jw; }
            else {
                const int i = max(0, d - nwj * k);         // tail bases in front of the region
                ls = src + nwj * k + i; t = tj + nwj + min(i, nt); nw = 0;
            }
            const int rank = lane + lo;
            tb.se_src[rank] = tb.rbase[lane] + (ls - c);
            tb.se_t[rank] = t;
            tb.se_nwin[rank] = nw;
            tb.reg_e0[lane] = rank;
        }
    }
    __syncwarp();
    // ---- halo: the 15 kept bases behind each region's last one, so a window that starts in a region reads on -------
    for (int idx = lane; idx < (NWC - 1) * HALO; idx += 32) {
        const int w = idx / HALO, i = idx - w * HALO;
        const int u = tb.cum[w + 1] + i;
        if (u < ktot) {
            const int s = slot_of(tb, u);
            const uint32_t dg = code_at(st, s, 1), fl = flags_at(st, s, 1);
            const int dst = tb.rbase[w] + (tb.cum[w + 1] - tb.cum[w]) + i;
            if (dg) atomicOr(&st[dst >> 4], dg << (30 - 2 * (dst & 15)));
            if (fl) atomicOr(&st[SW_CODE + (dst >> 5)], 1u << (31 - (dst & 31)));
        }
    }
    __syncwarp();
    return true;
}

// ---- per-token fallback emission of a tile with more record starts than the tables hold (all compute threads) -----
template <typename IdT, bool DENSE>
__device__ __noinline__ void emit_generic(const EncArgs &A, const uint32_t *st, const TileBuf &tb, int tid) {
    const EncParams &P = A.prm;
    const int k = P.k, m = tb.e_m, ktot = tb.ktot;
    const int64_t rlo = tb.e_rlo, t0 = (int64_t)tb.e_tile * A.S * TB, T0 = tb.T0;
    const int64_t *oo = A.out_off + rlo;
    auto kept = [&](int e) -> int { return DENSE ? (int)(rec_pos(A, rlo + e) - t0) : __ldcg(A.rec_k + rlo + e); };
    for (int j = tid; j < tb.ntok; j += NT) {
        int src, nwin, jj;
        if (j < tb.tok0) { src = -tb.pend; nwin = tb.nwin0; jj = j; }
        else {
            int lo = 0, hi = m;                            // last record start whose first token is at or before j
            while (hi - lo > 1) {
                const int mid = (lo + hi) >> 1;
                if (__ldcg(oo + mid) - T0 <= j) lo = mid; else hi = mid;
            }
            src = kept(lo);
            const int nxt = lo + 1 < m ? kept(lo + 1) : ktot;
            nwin = (int)div_k((uint32_t)(nxt - src), P);
            jj = j - (int)(__ldcg(oo + lo) - T0);
        }
        int32_t id;
        if (P.mode != MODE_KMER) {
            const uint32_t c = class_at(st, slot_of(tb, src + jj));
            id = c <= CLS_N ? P.nt_ids[c] : P.unk_id;
        } else if (jj < nwin) {
            uint32_t code = 0, bad = 0;
            for (int i = 0; i < k; ++i) {
                const int s = slot_of(tb, src + jj * k + i);
                code = (code << 2) | code_at(st, s, 1);
                bad |= flags_at(st, s, 1);
            }
            if (P.remap4) {
                uint32_t fl = 0;
                for (int i = 0; i < k; ++i) fl = (fl << 1) | flags_at(st, slot_of(tb, src + jj * k + i), 1);
                id = kmer_table_id_cold(P, code, fl, k);
            } else id = bad ? P.unk_id : (int32_t)(P.base_id + code);
        } else if (P.tail_policy == TAIL_PER_BASE) {
            const uint32_t c = class_at(st, slot_of(tb, src + nwin * k + (jj - nwin)));
            id = c <= CLS_N ? (P.remap4 ? P.nt_ids[c] : (int32_t)(P.base_id + P.four_k + c)) : P.unk_id;
        } else {
            id = P.unk_id;
        }
        store_id<IdT>(A, T0 + j, id);
    }
}

}  // namespace v7
}  // namespace dtk
