// encode_v7_compact.cuh -- the compute warps' byte loop: one region (S x 2 KiB) of a tile into the region's slice of
// the kept-base stream.  Included by encode_v7.cuh.
#pragma once

namespace dtk {
namespace v7 {

// byte q (0..63) of this lane's staged 64 bytes
__device__ __forceinline__ uint32_t staged_byte(const uint4 *slot, int q) {
    return reinterpret_cast<const uint8_t *>(slot)[q];
}

// ---- entry line state of a region, read off the 128 bytes in front of it when they settle it ---------------------
// (a newline or the record's start inside the window; always so for wrapped FASTA).  LS_UNKNOWN otherwise: the region
// then runs under the assumption IN_LINE and the scan warp checks it afterwards.
__device__ __noinline__ uint32_t region_entry_state(const EncArgs &A, const Smem7 &sm, const TileBuf &tb, int64_t t0, int64_t rs0,
                                                    int lane, int64_t pos_first, int64_t pos_last) {
    constexpr uint32_t FULL = 0xffffffffu;
    if (!A.prm.strip_headers) return LS_IN_LINE;
    if (rs0 <= pos_first || rs0 >= pos_last) return LS_LINE_START;          // no record byte on one side: irrelevant
    // start of the record that holds byte rs0 - 1, and whether a record starts right at rs0
    const int m = tb.m;
    const int64_t rlo = tb.rlo;
    int64_t prev;
    bool eq = false;
    if (m <= EV_MAX) {
        const int rel = (int)(rs0 - t0);
        int lt = 0;
        for (int b = 0; b < m; b += 32) {
            const int e = b + lane;
            const int p = e < m ? (int)tb.ev_p[e] : 0x7fffffff;
            lt += __popc(__ballot_sync(FULL, p < rel));
            eq = eq || __any_sync(FULL, p == rel);
            if (__any_sync(FULL, p >= rel)) break;
        }
        prev = lt > 0 ? t0 + tb.ev_p[lt - 1] : rec_pos(A, rlo - 1);
    } else {
        int64_t lo = rlo, hi = rlo + m;                                      // first record with position >= rs0
        while (lo < hi) {
            const int64_t mid = (lo + hi) >> 1;
            if (rec_pos(A, mid) >= rs0) hi = mid; else lo = mid + 1;
        }
        eq = lo < rlo + m && rec_pos(A, lo) == rs0;
        prev = rec_pos(A, lo - 1);
    }
    if (eq) return LS_LINE_START;                                            // a record starts right here
    uint32_t known = LS_UNKNOWN;
    const uint32_t wv = __ldg(reinterpret_cast<const uint32_t *>(A.bytes_al + rs0 - 128) + lane);
    uint32_t nlm = 0, nsk = 0, gtm = 0;                                      // bit i: byte i of this lane's word
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const uint32_t byte = (wv >> (8 * i)) & 255u;
        nlm |= (uint32_t)(byte == '\n') << i;
        gtm |= (uint32_t)(byte == '>') << i;
        nsk |= (uint32_t)(sm.lut[byte] != CLS_SKIP || byte == '>') << i;    // '>' opens a header even if the table skips it
    }
    int pstar = -1;                                                          // window index of the last line start
    const uint32_t nlb = __ballot_sync(FULL, nlm != 0);
    if (nlb) {
        const int L = 31 - __clz(nlb);
        const uint32_t mm = __shfl_sync(FULL, nlm, L);
        pstar = 4 * L + (31 - __clz(mm)) + 1;
    }
    const int64_t rsw = prev - (rs0 - 128);
    if (rsw >= 0 && rsw > pstar) pstar = (int)rsw;
    if (pstar >= 0) {
        uint32_t msk = nsk;
        const int lo = pstar - 4 * lane;                                     // this lane's bytes i >= lo count
        if (lo > 0) msk &= lo >= 4 ? 0u : (0xfu << lo);
        const uint32_t nb = __ballot_sync(FULL, msk != 0);
        if (!nb) known = LS_LINE_START;
        else {
            const int L = __ffs(nb) - 1;
            const uint32_t mm = __shfl_sync(FULL, msk, L), gg = __shfl_sync(FULL, gtm, L);
            known = ((gg >> (__ffs(mm) - 1)) & 1u) ? LS_IN_HEADER : LS_IN_LINE;
        }
    }
    return known;
}

// ---- general line-state step of one warp's 2 KiB (some lane holds a '>', a record start or a SKIP byte that is not
// a newline): per-lane summaries scanned over the warp, then the header mask of this lane's 64 bytes.  Out of line.
struct LsStep { unsigned long long hdr; uint32_t c_hr, c_x; };
__device__ __noinline__ LsStep line_state_step(unsigned long long nl, unsigned long long gt, unsigned long long osk,
                                               unsigned long long rs, uint32_t ls_in, int lane) {
    constexpr uint32_t FULL = 0xffffffffu;
    const unsigned long long ls_base = (nl >> 1) | rs;     // line starts: after each '\n' and at each record start
    auto settle = [&](unsigned long long ls, bool &pending) {   // move line starts over non-newline SKIP bytes
        pending = (nl & 1ull) != 0;
        unsigned long long t;
        while ((t = ls & osk) != 0) { pending = pending || (t & 1ull); ls = (ls & ~t) | (t >> 1); }
        return ls;
    };
    uint32_t s_hr, s_x;
    if ((gt | osk) == 0ull) {
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
        if (lane >= d) { s_x = ls_apply(s_hr, s_x, o_x); s_hr |= o_hr; }   // (earlier o) then (later s)
    }
    LsStep R;
    R.c_hr = __shfl_sync(FULL, s_hr, 31); R.c_x = __shfl_sync(FULL, s_x, 31);
    uint32_t e_hr = __shfl_up_sync(FULL, s_hr, 1), e_x = __shfl_up_sync(FULL, s_x, 1);
    if (lane == 0) { e_hr = 0; e_x = LS_LINE_START; }     // identity
    const uint32_t st_in = ls_apply(e_hr, e_x, ls_in);
    unsigned long long hdr = 0;
    if ((nl | gt | rs) == 0ull) {                         // no line ends or starts here: all header or none
        if (st_in == LS_IN_HEADER) hdr = ~0ull;
    } else if (gt == 0ull && st_in != LS_IN_HEADER) {
        // no '>' here and not inside a header: nothing of this lane's bytes is header
    } else {
        bool pd;
        const unsigned long long ls = settle(ls_base | (st_in == LS_LINE_START ? bit_at(0) : 0ull), pd);
        unsigned long long hs = ls & gt;                  // header lines that start inside this lane's bytes
        if (st_in == LS_IN_HEADER) {
            const int a = first_pos(nl), bb = first_pos(rs);
            const int e = (bb <= a) ? bb - 1 : a;         // through the '\n', or up to a record start
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
    R.hdr = hdr;
    return R;
}

// Record starts inside the 2 KiB that begin at position lo_pos, for a tile with more of them than the shared-memory
// list holds (records rlo .. rlo + m of rec_offsets): sets their bits in wk[32] (one 64-bit word per lane's bytes),
// returns how many there are and through e_lo the index of the first.  One warp, out of line (rare path).
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

// ---- append of one warp step to the region's stream slice ----------------------------------------------------------
// cst / fst: first code / flag word of the region; a = region-relative index of this lane's first kept base; n = its
// kept bases (planes compacted to the front, zero behind them).  The slice is zero beyond what was appended so far.
// Fast path (every lane holds >= 32 bases, so two lanes of equal parity never share a word): even lanes store, odd
// lanes read-modify-write; lane 0 merges with the word the previous step ended in.  Otherwise shared-memory atomics.
__device__ __forceinline__ void append_step(uint32_t *cst, uint32_t *fst, const uint32_t (&C)[4], unsigned long long bad,
                                            int a, int n, int lane) {
    constexpr uint32_t FULL = 0xffffffffu;
    const int cw0 = a >> 4, csh = 2 * (a & 15), cend = csh + 2 * n;      // code bits [csh, cend) of the words from cw0 on
    uint32_t cw[5];
    cw[0] = __funnelshift_r(C[0], 0u, csh);
    cw[1] = __funnelshift_r(C[1], C[0], csh);
    cw[2] = __funnelshift_r(C[2], C[1], csh);
    cw[3] = __funnelshift_r(C[3], C[2], csh);
    cw[4] = __funnelshift_r(0u, C[3], csh);
    const uint32_t bh = (uint32_t)(bad >> 32), bl = (uint32_t)bad;
    const int fw0 = a >> 5, fsh = a & 31, fend = fsh + n;
    uint32_t fw[3];
    fw[0] = __funnelshift_r(bh, 0u, fsh);
    fw[1] = __funnelshift_r(bl, bh, fsh);
    fw[2] = __funnelshift_r(0u, bl, fsh);
    uint32_t *cp = cst + cw0, *fp = fst + fw0;
    if (__all_sync(FULL, n >= 32)) {
        if (!(lane & 1)) {
            if (lane == 0) { if (csh) cw[0] |= cp[0]; if (fsh) fw[0] |= fp[0]; }
            cp[0] = cw[0]; cp[1] = cw[1];                        // n >= 32: at least 64 code bits and 32 flag bits
#pragma unroll
            for (int i = 2; i < 5; ++i) if (32 * i < cend) cp[i] = cw[i];
            fp[0] = fw[0];
#pragma unroll
            for (int i = 1; i < 3; ++i) if (32 * i < fend) fp[i] = fw[i];
        }
        __syncwarp();
        if (lane & 1) {
            cp[0] |= cw[0]; cp[1] |= cw[1];
#pragma unroll
            for (int i = 2; i < 5; ++i) if (32 * i < cend) cp[i] |= cw[i];
            fp[0] |= fw[0];
#pragma unroll
            for (int i = 1; i < 3; ++i) if (32 * i < fend) fp[i] |= fw[i];
        }
        __syncwarp();
    } else {
        if (n > 0) {
#pragma unroll
            for (int i = 0; i < 5; ++i) if (32 * i < cend && cw[i]) atomicOr(&cp[i], cw[i]);
#pragma unroll
            for (int i = 0; i < 3; ++i) if (32 * i < fend && fw[i]) atomicOr(&fp[i], fw[i]);
        }
        __syncwarp();
    }
}

// ---- one region ---------------------------------------------------------------------------------------------------
// The entry line state is read off the bytes in front of the region, or assumed IN_LINE when they do not settle it.
// The assumption can only be wrong inside a header line longer than that window; all it then costs is that the kept
// bases in front of the region's first line reset (hfix of them) must be dropped, which the scan warp does by moving
// the region's first slot -- no second pass.
template <bool DENSE>
__device__ __forceinline__ void compact_region(const EncArgs &A, Smem7 &sm, TileBuf &tb, uint32_t *st, int tile, int warp, int lane,
                                               int64_t pos_first, int64_t pos_last) {
    constexpr uint32_t FULL = 0xffffffffu;
    const EncParams &P = A.prm;
    const int S = A.S;
    const int RB = S * WB;
    const int64_t t0 = (int64_t)tile * S * TB;
    const int64_t rs0 = t0 + (int64_t)warp * RB;                 // position of the region's first byte
    uint32_t *const cst = st + (reg_slot(warp) >> 4);
    uint32_t *const fst = st + SW_CODE + (reg_slot(warp) >> 5);
    const int m = tb.m;
    const int64_t r_lo = tb.rlo;

    if (!DENSE) {
        // zero the slice (partial words are OR-ed in; the halo lands behind the last kept base)
        uint4 *c4 = reinterpret_cast<uint4 *>(cst), *f4 = reinterpret_cast<uint4 *>(fst);
        const int nc = (RB + 128) >> 6, nf = (RB + 128) >> 7;
        for (int i = lane; i < nc; i += 32) c4[i] = make_uint4(0, 0, 0, 0);
        for (int i = lane; i < nf; i += 32) f4[i] = make_uint4(0, 0, 0, 0);
    } else {
        // only the halo slots behind the region's RB bases are OR-ed into
        if (lane < 2) reinterpret_cast<uint4 *>(cst)[(RB >> 6) + lane] = make_uint4(0, 0, 0, 0);
        if (lane == 2) reinterpret_cast<uint4 *>(fst)[RB >> 7] = make_uint4(0, 0, 0, 0);
    }
    // line state carried along the region (warp-uniform) and the region's summary as a function of its entry state
    uint32_t ls = LS_IN_LINE, known = 1, r_hr = 0, r_x = LS_LINE_START;
    int hfix = -1;                                               // -1: no line reset seen yet
    if (!DENSE && P.strip_headers) {
        ls = region_entry_state(A, sm, tb, t0, rs0, lane, pos_first, pos_last);
        if (ls == LS_UNKNOWN) { known = 0; ls = LS_IN_LINE; }
    }
    const uint32_t ls_entry = ls;
    // record starts inside the region: events [ev, re_hi) of the tile's list (m <= EV_MAX)
    int ev = 0, re_hi = 0;
    if (!DENSE && m > 0 && m <= EV_MAX) {
        const int lo_rel = warp * RB, hi_rel = lo_rel + RB;
        for (int b = 0; b < m; b += 32) {
            const int e = b + lane;
            const int p = e < m ? (int)tb.ev_p[e] : 0x7fffffff;
            ev += __popc(__ballot_sync(FULL, p < lo_rel));
            re_hi += __popc(__ballot_sync(FULL, p < hi_rel));
        }
    }
    __syncwarp();
    int cnt = 0;                                                 // kept bases of the region so far
    uint4 *const slot = &sm.stage[warp][lane * 4];
    // everything inside the loop is region-relative and 32 bits wide (clamped where the 64-bit value is out of range)
    auto rel32 = [&](int64_t pos) -> int { const int64_t dlt = pos - rs0; return dlt < -(1 << 30) ? -(1 << 30) : (dlt > (1 << 30) ? (1 << 30) : (int)dlt); };
    const int end_rel = rel32(A.p_end), first_rel = rel32(pos_first), last_rel = rel32(pos_last);
    const uint4 *const src_lane = reinterpret_cast<const uint4 *>(A.bytes_al + rs0) + lane * 4;
#pragma unroll 1
    for (int s = 0; s < S; ++s) {
        const int w0r = s * WB;                                  // region offset of the warp's first byte
        const int p0r = w0r + lane * LB;                         //   and of this lane's
        if (w0r > end_rel) break;                                // (warp-uniform) nothing left; position p_end itself may hold the closing record offset
        uint4 v[4];
        {
            const uint4 *src = src_lane + s * (WB / 16);
            if (w0r + WB <= end_rel) {
#pragma unroll
                for (int j = 0; j < 4; ++j) v[j] = __ldg(src + j);
            } else {
#pragma unroll
                for (int j = 0; j < 4; ++j) v[j] = (p0r + 16 * j < end_rel) ? __ldg(src + j) : make_uint4(0, 0, 0, 0);
            }
        }
        uint32_t C[4];
        unsigned long long E;
        classify64(v, C, E);
        if (!P.fast_lut) E = ~0ull;
        unsigned long long bad = E;
        // runs of N: classified arithmetically too (their digit is already 2), not one LUT trip per byte
        if (P.fast_lut && P.fast_n && __any_sync(FULL, __popcll(E) >= 4)) E &= ~n_plane(v[0], v[1], v[2], v[3]);
        // first trip through the LUT for every byte still flagged: what the line state and the keep mask need, and
        // which bytes need their digit / flag corrected if they are kept
        unsigned long long skip = 0, nl = 0, gt = 0, fix = 0;
        if (E) {
#pragma unroll
            for (int j = 0; j < 4; ++j) slot[j] = v[j];         // (bank conflicts cost LSU cycles, which are plentiful; a swizzle costs ALU)
            unsigned long long rem = E;
            while (rem) {
                const int q = __clzll((long long)rem);
                const unsigned long long bq = bit_at(q);
                rem ^= bq;
                const uint32_t byte = staged_byte(slot, q);
                const uint32_t c = sm.lut[byte];
                if (byte == '\n') nl |= bq;
                if (byte == '>') gt |= bq;
                if (c == CLS_SKIP) skip |= bq;
                else if (!(c == CLS_N && (byte | 0x20u) == 'n' && P.fast_lut)) fix |= bq;
            }
        }
        int n = LB, a;
        if (DENSE) {
            // every byte is a kept base at its own position: correct the flagged ones in place
            unsigned long long rem = fix;
            while (rem) {
                const int q = __clzll((long long)rem);
                const unsigned long long bq = bit_at(q);
                rem ^= bq;
                const uint32_t c = sm.lut[staged_byte(slot, q)];
                if (c < CLS_N) bad &= ~bq;
                set_digit(C, q, c < CLS_N ? c : (c == CLS_N ? 2u : 1u));
            }
            a = s * WB + lane * LB;
            *reinterpret_cast<uint4 *>(cst + (a >> 4)) = make_uint4(C[0], C[1], C[2], C[3]);
            *reinterpret_cast<uint2 *>(fst + (a >> 5)) = make_uint2((uint32_t)(bad >> 32), (uint32_t)bad);
            continue;
        }
        // ---- record starts inside this warp's 2 KiB (rare) ----------------------------------------------------------
        int e_lo = 0, e_cnt = 0;
        unsigned long long rs = 0ull;
        const int wrel = warp * RB + s * WB;                     // tile position of the warp's first byte
        if (m > 0) {
            if (m <= EV_MAX) {
                if (ev < re_hi && (int)tb.ev_p[ev] < wrel + WB) {          // (warp-uniform)
                    e_lo = ev;
                    sm.wk[warp][lane] = 0ull;
                    __syncwarp();
                    for (;;) {
                        const int e = ev + lane;
                        const int p = e < re_hi ? (int)tb.ev_p[e] - wrel : WB;
                        const uint32_t inr = __ballot_sync(FULL, p < WB);
                        if (p < WB) atomicOr(&sm.wk[warp][p >> 6], bit_at(p & 63));
                        ev += __popc(inr);
                        if (inr != FULL) break;
                    }
                    e_cnt = ev - e_lo;
                    __syncwarp();
                    rs = sm.wk[warp][lane];
                }
            } else {
                e_cnt = warp_events_many(A, sm.wk[warp], r_lo, m, rs0 + w0r, lane, e_lo);
                if (e_cnt) { __syncwarp(); rs = sm.wk[warp][lane]; }
            }
        }
        // ---- line state and header mask -----------------------------------------------------------------------------
        unsigned long long hdr = 0;
        bool first_reset = false;                                // (warp-uniform) the region's first line reset is in this step
        if (P.strip_headers) {
            const unsigned long long osk = skip & ~nl & ~gt;     // SKIP bytes that neither end nor start a line
            uint32_t c_hr, c_x;
            if (!__any_sync(FULL, (gt | rs | osk) != 0ull)) {
                // no '>', no record start, no odd SKIP byte in these 2 KiB: a header can only run on from before
                const uint32_t nlb = __ballot_sync(FULL, nl != 0ull);
                if (ls == LS_IN_HEADER) {
                    const int first = nlb ? __ffs(nlb) - 1 : 32;
                    if (lane < first) hdr = ~0ull;
                    else if (lane == first) { const int e = first_pos(nl); hdr = e >= 63 ? ~0ull : ~from_pos(e + 1); }
                }
                c_hr = nlb != 0u;
                c_x = (__shfl_sync(FULL, (uint32_t)nl, 31) & 1u) ? LS_LINE_START : LS_IN_LINE;
            } else {
                const LsStep R = line_state_step(nl, gt, osk, rs, ls, lane);
                hdr = R.hdr; c_hr = R.c_hr; c_x = R.c_x;
            }
            ls = ls_apply(c_hr, c_x, ls);
            first_reset = !known && hfix < 0 && c_hr;
            r_x = ls_apply(c_hr, c_x, r_x); r_hr |= c_hr;
        }
        unsigned long long keep = ~skip & ~hdr;
        if (p0r < first_rel || p0r + LB > last_rel) {
            const int ia = first_rel - p0r, ib = last_rel - p0r;         // in-record positions are [ia, ib)
            const unsigned long long ma = ia <= 0 ? ~0ull : from_pos(ia > 64 ? 64 : ia);
            const unsigned long long mb = ib <= 0 ? 0ull : (ib >= 64 ? ~0ull : ~from_pos(ib));
            keep &= ma & mb;
        }
        {
            // second trip: digit and flag of every kept byte the arithmetic did not get right
            unsigned long long rem = fix & keep;
            while (rem) {
                const int q = __clzll((long long)rem);
                const unsigned long long bq = bit_at(q);
                rem ^= bq;
                const uint32_t c = sm.lut[staged_byte(slot, q)];
                if (c < CLS_N) bad &= ~bq;
                set_digit(C, q, c < CLS_N ? c : (c == CLS_N ? 2u : 1u));
            }
        }
        // ---- delete what is dropped, warp prefix of the kept counts -------------------------------------------------
        n = __popcll(keep);
        if (n == 63) delete_one(C, bad, __clzll((long long)~keep));
        else if (n == 0) { C[0] = C[1] = C[2] = C[3] = 0u; bad = 0ull; }
        else if (n != 64) delete_runs(C, bad, keep);
        int total;
        if (__all_sync(FULL, n >= 63)) {
            const uint32_t miss = __ballot_sync(FULL, n == 63);
            a = LB * lane - __popc(miss & ((1u << lane) - 1u));
            total = WB - __popc(miss);
        } else {
            int inc = n;
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) { const int t = __shfl_up_sync(FULL, inc, d); if (lane >= d) inc += t; }
            a = inc - n;
            total = __shfl_sync(FULL, inc, 31);
        }
        append_step(cst, fst, C, bad, cnt + a, n, lane);
        if (first_reset) {
            // kept bases (under the IN_LINE assumption) in front of the first '\n' or record start of the region
            const unsigned long long rz = nl | rs;
            const int L = __ffs(__ballot_sync(FULL, rz != 0ull)) - 1;
            const int q = first_pos(rz);
            hfix = cnt + __shfl_sync(FULL, a + (q ? __popcll(keep >> (64 - q)) : 0), L);
        }
        if (e_cnt) {                                             // (warp-uniform) kept bases in front of each record start
            sm.wk[warp][lane] = keep; sm.offw[warp][lane] = (uint16_t)a;
            __syncwarp();
            for (int e = e_lo + lane; e < e_lo + e_cnt; e += 32) {
                const int p = (m <= EV_MAX ? (int)tb.ev_p[e] : (int)(rec_pos(A, r_lo + e) - t0)) - wrel;
                const int o = p >> 6, q = p & 63;
                const int kidx = cnt + (int)sm.offw[warp][o] + (q ? __popcll(sm.wk[warp][o] >> (64 - q)) : 0);
                if (m <= EV_MAX) tb.ev_k[e] = kidx | (warp << 16); else A.rec_k[r_lo + e] = kidx | (warp << 16);
            }
            __syncwarp();
        }
        cnt += total;
    }
    if (lane == 0) {
        tb.reg_cnt[warp] = DENSE ? RB : cnt;
        tb.reg_hfix[warp] = hfix < 0 ? cnt : hfix;
        tb.reg_ls[warp] = (known << 8) | (ls_entry << 4) | (r_hr << 2) | r_x;
    }
}

}  // namespace v7
}  // namespace dtk
