// encode_v7_kernel.cuh -- the persistent kernel: role split and hand-offs.  Included by encode_v7.cuh.
#pragma once

namespace dtk {
namespace v7 {

#ifdef DTK_PROF
#define PROF_T(var) const long long var = clock64()
#define PROF_ADD(slot, t0, t1) do { if (lane == 0) atomicAdd(&A.prof[slot], (unsigned long long)((t1) - (t0))); } while (0)
#define PROF_INC(slot) do { if (lane == 0) atomicAdd(&A.prof[slot], 1ull); } while (0)
#else
#define PROF_T(var)
#define PROF_ADD(slot, t0, t1)
#define PROF_INC(slot)
#endif

// KK: the emission variant compiled in -- 0 single-nt, 1..6 / 8 that k, -1 every variant behind a run-time switch.
// Loop iteration i of a CTA:   compute warps: compact tile B_i -> DONE -> (READY) emit tile B_{i-1}
//                              scan warp:     prefix + tables of B_{i-1} -> READY || (DONE) aggregate of B_i; then prepare B_{i+1} -> PREP
template <typename IdT, int KK, bool DENSE>
__global__ void __launch_bounds__(NT7, 3) encode_tiles_v7(const __grid_constant__ EncArgs A) {
    extern __shared__ __align__(16) uint8_t smem_raw[];
    Smem7 &sm = *reinterpret_cast<Smem7 *>(smem_raw);
    constexpr uint32_t FULL = 0xffffffffu;
    const EncParams &P = A.prm;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int64_t pos_first = rec_pos(A, 0), pos_last = rec_pos(A, A.n_rec);   // bytes outside are in no record

    if (tid < 256) sm.lut[tid] = A.lut[tid];
    // launched with programmatic stream serialisation: everything above overlaps the tail of the pre-pass kernel, whose
    // outputs (first_rec, out_offsets) are read only behind this point (a no-op in an ordinary launch)
    // ... and so does the fetch of the tile this CTA will most likely draw first (tickets go out in launch order), as a hint
    // to L2: the input bytes are nobody's output, and HBM idles while the pre-pass runs
    if (tid < A.S) {
        const int64_t p0 = ((int64_t)blockIdx.x * A.S + tid) * TB;
        int64_t sz = A.p_end - p0; if (sz > TB) sz = TB; sz &= ~(int64_t)15;
        if (sz > 0) asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(A.bytes_al + p0), "r"((uint32_t)sz) : "memory");
    }
    asm volatile("griddepcontrol.wait;" ::: "memory");
    if (tid == 0) sm.done_cnt = 0;
    __syncthreads();

    if (warp == NWC) {
        // =============================================== scan warp ===================================================
        // Iteration i of the compute warps compacts tile B_i and then emits B_{i-1}; the scan warp runs one message
        // ahead: PREP(i+1) goes out at the start of iteration i, so the compute warps never wait for a sibling warp or
        // for this warp between tiles -- only READY(i) needs every region of B_{i-1} (finished a whole tile ago).
        unsigned long long ticket = 0;
        if (lane == 0) ticket = atomicAdd(A.ticket, 1ull);
        ticket = __shfl_sync(FULL, ticket, 0);
        int bufB = 0;
        int tileB = scan_prep(A, sm.tb[0], ticket, lane);
        if (lane == 0) {
            TileCtl &c = sm.ctl[0];
            c.tile = tileB; c.buf = 0; c.emit = 0; c.emit_buf = 0; c.emit_generic = 0; c.last = tileB < 0;
        }
        __threadfence_block();
        bar_arrive(BAR_PREP);
        bool pendA = false;                                // the tile in bufB ^ 1 still waits for its prefix + tables
        bool force = false;
        int done_target = 0, spins = 0, it = 0;
        auto stuck = [&]() {                               // bounded wait: a broken chain sets the status word instead of hanging
            if (++spins > SPIN_LIMIT / 4) { if (lane == 0) A.status[1] = 1u; force = true; }
            __nanosleep(64);
        };
#pragma unroll 1
        for (; tileB >= 0; ++it) {
            TileBuf &tbB = sm.tb[bufB];
            if (pendA && scan_tables<DENSE>(A, sm, sm.tb[bufB ^ 1], sm.strm[bufB ^ 1], lane, force)) {
                __threadfence_block();
                bar_arrive(BAR_READY + (it & 1));
                pendA = false;
            }
            // ---- next tile into the other buffer (the preparation only touches tile / m / rlo / ev_p, which neither
            //      the tables nor the emission of the tile held there read any more)
            PROF_T(p0);
            if (lane == 0) ticket = atomicAdd(A.ticket, 1ull);
            ticket = __shfl_sync(FULL, ticket, 0);
            const int tileC = scan_prep(A, sm.tb[bufB ^ 1], ticket, lane);
            PROF_T(p1); PROF_ADD(0, p0, p1);
            if (lane == 0) {
                TileCtl &nx = sm.ctl[(it + 1) & 1];
                nx.tile = tileC; nx.buf = bufB ^ 1; nx.emit = 1; nx.emit_buf = bufB; nx.emit_generic = tbB.m > EV_MAX; nx.last = tileC < 0;
            }
            __threadfence_block();
            bar_arrive(BAR_PREP + ((it + 1) & 1));
            // ---- two jobs, neither of which may hold up the other: prefix + tables of the tile to emit (needs the
            //      predecessors' aggregates), aggregate of the tile being compacted (needs the compute warps)
            PROF_T(p2);
            for (bool needD = true; pendA || needD;) {
                bool progress = false;
                if (pendA && scan_tables<DENSE>(A, sm, sm.tb[bufB ^ 1], sm.strm[bufB ^ 1], lane, force)) {
                    __threadfence_block();
                    bar_arrive(BAR_READY + (it & 1));
                    pendA = false; progress = true;
                }
                if (needD && *(volatile int32_t *)&sm.done_cnt >= done_target + NWC) {
                    __threadfence_block();
                    done_target += NWC;
                    PROF_T(a0);
                    scan_regions<DENSE>(A, tbB, lane);
                    scan_aggregate<DENSE>(A, tbB, sm.strm[bufB], lane);
                    PROF_T(a1); PROF_ADD(2, a0, a1);
                    needD = false; progress = true;
                }
                if (!progress) stuck(); else spins = 0;
            }
            // ---- the tile just aggregated gets its prefix right away: the sooner its inclusive prefix is out, the
            //      shorter every successor's walk back (its emission is a whole tile away)
            PROF_T(p3); PROF_ADD(1, p2, p3);
            if (scan_tables<DENSE>(A, sm, tbB, sm.strm[bufB], lane, force)) {
                __threadfence_block();
                bar_arrive(BAR_READY + ((it + 1) & 1));
            } else { pendA = true; PROF_INC(4); }
            PROF_T(p4); PROF_ADD(3, p3, p4); PROF_INC(5);
            tileB = tileC; bufB ^= 1;
        }
        if (pendA) {
            while (!scan_tables<DENSE>(A, sm, sm.tb[bufB ^ 1], sm.strm[bufB ^ 1], lane, force)) stuck();
            __threadfence_block();
            bar_arrive(BAR_READY + (it & 1));
        }
        return;
    }

    // ================================================= compute warps ====================================================
    const bool affine = P.nt_ids[1] == P.nt_ids[0] + 1 && P.nt_ids[2] == P.nt_ids[0] + 2 && P.nt_ids[3] == P.nt_ids[0] + 3;
    const bool vec_ok = (reinterpret_cast<uintptr_t>(A.ids) & 15) == 0 &&
                        (P.mode != MODE_KMER || (P.k >= 1 && P.k <= 6) || P.k == 8);
#pragma unroll 1
    for (int it = 0;; ++it) {
        PROF_T(c0);
        bar_sync(BAR_PREP + (it & 1));
        PROF_T(c1); if (warp == 0) PROF_ADD(8, c0, c1);
        const TileCtl &c = sm.ctl[it & 1];
        const int tile = c.tile, buf = c.buf, emit = c.emit, ebuf = c.emit_buf, egen = c.emit_generic, last = c.last;
        if (tile >= 0) {
            compact_region<DENSE>(A, sm, sm.tb[buf], sm.strm[buf], tile, warp, lane, pos_first, pos_last);
            __syncwarp();
            if (lane == 0) { __threadfence_block(); atomicAdd(&sm.done_cnt, 1); }
        }
        PROF_T(c2); if (warp == 0) PROF_ADD(9, c1, c2);
        if (emit) {
            bar_sync(BAR_READY + (it & 1));
            PROF_T(c3); if (warp == 0) PROF_ADD(10, c2, c3);
            const TileBuf &ta = sm.tb[ebuf];
            if (egen) emit_generic<IdT, DENSE>(A, sm.strm[ebuf], ta, tid);
            else emit_region<IdT, KK>(A, sm.strm[ebuf], ta, warp, lane, vec_ok, affine);
            PROF_T(c4); if (warp == 0) PROF_ADD(11, c3, c4);
        }
        if (last) break;
    }
}

}  // namespace v7
}  // namespace dtk
