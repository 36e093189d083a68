// pad_kernel.cuh -- padding / attention-mask writer.
//
// Row r of batch_ids[n_rows][seq_len] gets record r's first m = min(tokens, seq_len) ids;
// LEFT padding right-aligns them (Alg. 2 l.12-14: "left-pad each row with
// id_pad, right-aligning the original T positions"), RIGHT padding left-aligns them; every
// other column holds pad_id; mask is 1 exactly on the m kept columns (Q14-Q16).
// Pure write traffic: 5 bytes out per column, <= 4 (or 2) bytes in per kept column.
#pragma once
#include "common.cuh"

namespace dtk {

struct PadArgs {
    const void *ids;
    const int64_t *out_off;
    int64_t n_rows;
    int32_t *batch_ids;
    uint8_t *mask;              // may be null
    int32_t seq_len, pad_side, pad_id;
    int64_t ids_cap;            // ids beyond it were never written (an encode that overflowed): read as pad_id
    const uint32_t *run_if;     // non-null: the kernel returns at once unless *run_if != 0 (the fused path's fall-back)
};

// one CTA per row (grid-stride), each thread writes 4 consecutive columns per step
template <typename IdT>
__global__ void __launch_bounds__(256) pad_rows_kernel(const __grid_constant__ PadArgs A) {
    if (A.run_if && *A.run_if == 0u) return;
    const IdT *ids = reinterpret_cast<const IdT *>(A.ids);
    const int L = A.seq_len;
    // 16-byte id stores and 4-byte mask stores need aligned rows: seq_len a multiple of 4 and aligned base pointers
    const bool vec = (L & 3) == 0 && (reinterpret_cast<uintptr_t>(A.batch_ids) & 15) == 0 &&
                     (reinterpret_cast<uintptr_t>(A.mask) & 3) == 0;
    for (int64_t r = blockIdx.x; r < A.n_rows; r += gridDim.x) {
        const int64_t o0 = A.out_off[r];
        const int64_t tok = A.out_off[r + 1] - o0;
        const int m = (int)(tok < L ? tok : L);
        const int col0 = (A.pad_side == 0) ? L - m : 0;          // first kept column
        int32_t *row = A.batch_ids + r * L;
        uint8_t *mrow = A.mask ? A.mask + r * L : nullptr;
        if (vec) {
            for (int c = threadIdx.x * 4; c < L; c += blockDim.x * 4) {
                int4 v; uint32_t mk = 0;
                int32_t *pv = reinterpret_cast<int32_t *>(&v);
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    int q = c + j - col0;
                    bool in = q >= 0 && q < m;
                    pv[j] = (in && o0 + q < A.ids_cap) ? (int32_t)ids[o0 + q] : A.pad_id;
                    mk |= (uint32_t)in << (8 * j);
                }
                *reinterpret_cast<int4 *>(row + c) = v;
                if (mrow) *reinterpret_cast<uint32_t *>(mrow + c) = mk;
            }
        } else {
            for (int c = threadIdx.x; c < L; c += blockDim.x) {
                int q = c - col0;
                bool in = q >= 0 && q < m;
                row[c] = (in && o0 + q < A.ids_cap) ? (int32_t)ids[o0 + q] : A.pad_id;
                if (mrow) mrow[c] = in ? 1 : 0;
            }
        }
    }
}

}  // namespace dtk
