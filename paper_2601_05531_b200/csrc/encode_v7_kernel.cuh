// encode_v7_kernel.cuh -- the persistent kernel: role split and hand-offs.  Included by encode_v7.cuh.
#pragma once

namespace dtk {

// KK: the emission variant compiled in -- 0 single-nt, 1..6 / 8 that k, -1 every variant behind a run-time switch.
// Loop iteration i of a CTA:   compute warps: compact tile B_i -> DONE -> (READY) emit tile B_{i-1}
//                              scan warp:     prefix + tables of B_{i-1} -> READY; (DONE) aggregate of B_i; prepare B_{i+1} -> PREP
template <typename IdT, int KK, bool DENSE>
__global__ void __launch_bounds__(NT7, 3) encode_tiles_v7(const __grid_constant__ EncArgs A) {
    extern __shared__ __align__(16) uint8_t smem_raw[];
    Smem7 &sm = *reinterpret_cast<Smem7 *>(smem_raw);
    constexpr uint32_t FULL = 0xffffffffu;
    const EncParams &P = A.prm;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int64_t pos_first = rec_pos(A, 0), pos_last = rec_pos(A, A.n_rec);   // bytes outside are in no record

    if (tid < 256) sm.lut[tid] = A.lut[tid];
    __syncthreads();

    if (warp == NWC) {
        // =============================================== scan warp ===================================================
        unsigned long long ticket = 0;
        if (lane == 0) ticket = atomicAdd(A.ticket, 1ull);
        ticket = __shfl_sync(FULL, ticket, 0);
        int bufB = 0;
        int tileB = scan_prep(A, sm.tb[bufB], ticket, lane);
        if (lane == 0) {
            TileCtl &c = sm.ctl[0];
            c.tile = tileB; c.buf = bufB; c.emit = 0; c.emit_buf = 0; c.emit_generic = 0; c.redo = 0; c.last = tileB < 0;
        }
        __threadfence_block();
        bar_arrive(BAR_PREP);
        if (tileB >= 0) {
            if (lane == 0) ticket = atomicAdd(A.ticket, 1ull);
            ticket = __shfl_sync(FULL, ticket, 0);
        }
        bool emitA = false;                                // this iteration ends with the emission of the tile in bufB ^ 1
        int rdy = 0;                                       // READY alternates between two barrier ids
#pragma unroll 1
        for (int it = 0; tileB >= 0 || emitA; ++it) {
            TileCtl &nx = sm.ctl[(it + 1) & 1];
            if (emitA) {
                TileBuf &ta = sm.tb[bufB ^ 1];
                scan_tables<DENSE>(A, sm, ta, sm.strm[bufB ^ 1], lane);
                __threadfence_block();
                bar_arrive(BAR_READY + rdy);
                rdy ^= 1;
            }
            if (tileB < 0) break;                          // that was the last emission
            bar_sync(BAR_DONE);
            TileBuf &tbB = sm.tb[bufB];
            uint32_t ent[NWC];
            if (scan_regions<DENSE>(A, tbB, lane, ent)) {
                // some region assumed a wrong entry line state: the compute warps go over the tile again
                if (lane == 0) {
                    nx.tile = tileB; nx.buf = bufB; nx.emit = 0; nx.emit_buf = 0; nx.emit_generic = 0; nx.redo = 1; nx.last = 0;
#pragma unroll
                    for (int w = 0; w < NWC; ++w) nx.ent_ls[w] = ent[w];
                }
                __threadfence_block();
                bar_arrive(BAR_PREP);
                emitA = false;
                continue;
            }
            scan_aggregate<DENSE>(A, tbB, sm.strm[bufB], lane);
            // next tile into the other buffer
            const int tileC = scan_prep(A, sm.tb[bufB ^ 1], ticket, lane);   // (its tables were last read two iterations ago)
            if (lane == 0) {
                nx.tile = tileC; nx.buf = bufB ^ 1; nx.emit = 1; nx.emit_buf = bufB; nx.emit_generic = tbB.m > EV_MAX; nx.redo = 0; nx.last = tileC < 0;
            }
            __threadfence_block();
            bar_arrive(BAR_PREP);
            if (tileC >= 0) {
                if (lane == 0) ticket = atomicAdd(A.ticket, 1ull);
                ticket = __shfl_sync(FULL, ticket, 0);
            }
            tileB = tileC; bufB ^= 1; emitA = true;
        }
        return;
    }

    // ================================================= compute warps ====================================================
    const bool affine = P.nt_ids[1] == P.nt_ids[0] + 1 && P.nt_ids[2] == P.nt_ids[0] + 2 && P.nt_ids[3] == P.nt_ids[0] + 3;
    const bool vec_ok = (reinterpret_cast<uintptr_t>(A.ids) & 15) == 0 &&
                        (P.mode != MODE_KMER || (P.k >= 1 && P.k <= 6) || P.k == 8);
    int rdy = 0;
#pragma unroll 1
    for (int it = 0;; ++it) {
        bar_sync(BAR_PREP);
        const TileCtl &c = sm.ctl[it & 1];
        const int tile = c.tile, buf = c.buf, emit = c.emit, ebuf = c.emit_buf, egen = c.emit_generic, last = c.last;
        if (tile >= 0) {
            compact_region<DENSE>(A, sm, sm.tb[buf], sm.strm[buf], tile, warp, lane, c.redo != 0, c.ent_ls[warp], pos_first, pos_last);
            __threadfence_block();
            bar_arrive(BAR_DONE);
        }
        if (emit) {
            bar_sync(BAR_READY + rdy);
            rdy ^= 1;
            const TileBuf &ta = sm.tb[ebuf];
            if (egen) emit_generic<IdT, DENSE>(A, sm.strm[ebuf], ta, tid);
            else emit_region<IdT, KK>(A, sm.strm[ebuf], ta, warp, lane, vec_ok, affine);
        }
        if (last) break;
    }
}

}  // namespace dtk
