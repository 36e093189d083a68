// ext_kernels.cuh -- the SURVEY.md 8(f) operations that sit next to the encoder: reverse complement and decode
// (PAPER.md:315-317, 325-327), the embedding gather behind the paper's micro-batch rule,
// and the int32 -> int64 widening of the paper's IDs path.  All are plain streaming kernels bound by
// HBM: 16-byte accesses on the wide side, grid-stride loops, no shared state between calls.
#pragma once
#include "common.cuh"

namespace dtk {

// ---- reverse complement ---------------------------------------------------------------------------------------
// Complement of every byte value: A<->T, C<->G, U->A, IUPAC R<->Y, K<->M, B<->V, D<->H; S, W, N and every other byte
// map to themselves; case is kept.
__device__ __forceinline__ uint32_t comp_byte(uint32_t b) {
    const uint32_t up = b & 0xDFu, lowbit = b & 0x20u;
    if (up < 'A' || up > 'Y') return b;
    // "ABCDEFGHIJKLMNOPQRSTUVWXY" -> complement (letters without one map to themselves)
    const char *t = "TVGHEFCDIJMLKNOPQYSAABWXR";
    return (uint32_t)(uint8_t)t[up - 'A'] | lowbit;
}

struct RevcompArgs {
    const uint8_t *in; uint8_t *out;
    const int64_t *rec_off; int64_t n_rec, n_bytes;
};

// One thread per 16 output bytes.  The record of the first byte comes from a binary search of rec_offsets; the
// source bytes of a record's output position p are read from the mirrored position start + end - 1 - p.
__global__ void __launch_bounds__(256) revcomp_kernel(const __grid_constant__ RevcompArgs A) {
    __shared__ uint8_t tab[256];
    tab[threadIdx.x] = (uint8_t)comp_byte(threadIdx.x);
    __syncthreads();
    const int64_t n16 = (A.n_bytes + 15) >> 4;
    const bool vec = ((reinterpret_cast<uintptr_t>(A.out) & 15) == 0);
    for (int64_t g = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; g < n16; g += (int64_t)gridDim.x * blockDim.x) {
        const int64_t p0 = g << 4;
        // r = last record with rec_off[r] <= p0 (or -1)
        int64_t lo = 0, hi = A.n_rec + 1;
        while (lo < hi) { const int64_t mid = (lo + hi) >> 1; if (A.rec_off[mid] <= p0) lo = mid + 1; else hi = mid; }
        int64_t r = lo - 1;
        int64_t a = r >= 0 ? A.rec_off[r] : 0, e = (r >= 0 && r < A.n_rec) ? A.rec_off[r + 1] : (r < 0 ? A.rec_off[0] : A.n_bytes);
        bool inrec = r >= 0 && r < A.n_rec;
        uint32_t w[4] = {0u, 0u, 0u, 0u};
        const int nb = (int)min((int64_t)16, A.n_bytes - p0);
        for (int x = 0; x < nb; ++x) {
            const int64_t p = p0 + x;
            while (p >= e && r < A.n_rec) {                      // next record (empty ones are skipped)
                ++r;
                inrec = r < A.n_rec;
                a = e; e = inrec ? A.rec_off[r + 1] : A.n_bytes;
                if (inrec) a = A.rec_off[r];
            }
            const uint32_t b = (inrec && p >= a) ? (uint32_t)tab[A.in[a + e - 1 - p]] : (uint32_t)A.in[p];   // outside every record: copied
            w[x >> 2] |= b << (8 * (x & 3));
        }
        if (vec && nb == 16) *reinterpret_cast<uint4 *>(A.out + p0) = make_uint4(w[0], w[1], w[2], w[3]);
        else for (int x = 0; x < nb; ++x) A.out[p0 + x] = (uint8_t)(w[x >> 2] >> (8 * (x & 3)));
    }
}

// ---- decode ---------------------------------------------------------------------------------------------------
struct DecodeArgs {
    const void *ids; const int64_t *out_off; int64_t n_rec;
    int32_t mode, k, base_id, n_id, pad_id;
    int32_t nt_ids[5];
    int64_t four_k;
    int32_t n_tokens_bpe;          // 4 + n_merges
    const uint32_t *spell_off;     // BPE: [n_tokens_bpe + 1] offsets into spell
    const uint8_t *spell;          // BPE: spellings of all tokens, back to back
    int32_t *rec_len;              // [n_rec] decoded bytes per record
    const int64_t *byte_off;       // [n_rec + 1] (write pass)
    uint8_t *out; int64_t out_cap;
    uint32_t *status;
};

// bytes the token spells (0 for pad_id)
__device__ __forceinline__ int decode_len(const DecodeArgs &A, int32_t id) {
    if (id == A.pad_id) return 0;
    if (A.mode == MODE_SINGLE_NT) return 1;
    if (A.mode == MODE_KMER) {
        const int64_t code = (int64_t)id - A.base_id;
        return (code >= A.four_k && code < A.four_k + 5) ? 1 : A.k;
    }
    const int64_t t = (int64_t)id - A.base_id;
    if (id == A.n_id || t < 0 || t >= A.n_tokens_bpe) return 1;
    return (int)(A.spell_off[t + 1] - A.spell_off[t]);
}

// WRITE = false: decoded length of every record.  WRITE = true: the bytes, at byte_off[r] + prefix inside the record.
// One warp per record, 32 tokens per step.
template <typename IdT, bool WRITE>
__global__ void __launch_bounds__(256) decode_kernel(const __grid_constant__ DecodeArgs A) {
    constexpr uint32_t FULL = 0xffffffffu;
    const int lane = threadIdx.x & 31;
    const int64_t warp = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int64_t nwarps = ((int64_t)gridDim.x * blockDim.x) >> 5;
    const IdT *ids = reinterpret_cast<const IdT *>(A.ids);
    for (int64_t r = warp; r < A.n_rec; r += nwarps) {
        const int64_t t0 = A.out_off[r], t1 = A.out_off[r + 1];
        int64_t pos = WRITE ? A.byte_off[r] : 0;
        for (int64_t base = t0; base < t1; base += 32) {
            const int64_t j = base + lane;
            const int32_t id = j < t1 ? (int32_t)ids[j] : A.pad_id;
            const int len = j < t1 ? decode_len(A, id) : 0;
            int inc = len;
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) { const int t = __shfl_up_sync(FULL, inc, d); if (lane >= d) inc += t; }
            if (WRITE && len > 0) {
                const int64_t at = pos + inc - len;
                if (at + len > A.out_cap) { A.status[0] = 1u; }
                else if (A.mode == MODE_SINGLE_NT) {
                    uint8_t ch = 'N';
#pragma unroll
                    for (int c = 0; c < 5; ++c) if (id == A.nt_ids[c]) { ch = (uint8_t)"ACGTN"[c]; break; }
                    A.out[at] = ch;
                } else if (A.mode == MODE_KMER) {
                    const int64_t code = (int64_t)id - A.base_id;
                    if (code >= 0 && code < A.four_k) {
                        for (int i = 0; i < A.k; ++i) A.out[at + i] = (uint8_t)"ACGT"[(code >> (2 * (A.k - 1 - i))) & 3];
                    } else if (code >= A.four_k && code < A.four_k + 5) {
                        A.out[at] = (uint8_t)"ACGTN"[code - A.four_k];
                    } else {
                        for (int i = 0; i < A.k; ++i) A.out[at + i] = 'N';
                    }
                } else {
                    const int64_t t = (int64_t)id - A.base_id;
                    if (id == A.n_id || t < 0 || t >= A.n_tokens_bpe) A.out[at] = 'N';
                    else {
                        const uint8_t *s = A.spell + A.spell_off[t];
                        for (int i = 0; i < len; ++i) A.out[at + i] = s[i];
                    }
                }
            }
            pos += __shfl_sync(FULL, inc, 31);
        }
        if (!WRITE && lane == 0) A.rec_len[r] = (int32_t)pos;
    }
}

// ---- embedding gather -----------------------------------------------------------------------------------------
// out[i][:] = table[ids[i]][:] for tokens i in [0, n_tokens), rows of row_bytes bytes; an ID outside [0, vocab) gives
// a zero row.  VEC = bytes per access (16 or 4); one thread per access, consecutive threads write consecutive bytes.
template <int VEC>
__global__ void __launch_bounds__(256) embed_kernel(const int32_t *ids, int64_t n_tokens, const uint8_t *table, int64_t vocab,
                                                    int32_t row_bytes, uint8_t *out) {
    const int per = row_bytes / VEC;                       // accesses per row
    const int64_t total = n_tokens * per;
    for (int64_t g = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; g < total; g += (int64_t)gridDim.x * blockDim.x) {
        const int64_t tok = g / per;
        const int piece = (int)(g - tok * per);
        const int32_t id = __ldg(ids + tok);
        const bool ok = id >= 0 && id < vocab;
        if (VEC == 16) {
            uint4 v = make_uint4(0u, 0u, 0u, 0u);
            if (ok) v = __ldg(reinterpret_cast<const uint4 *>(table + (int64_t)id * row_bytes) + piece);
            reinterpret_cast<uint4 *>(out)[g] = v;
        } else {
            uint32_t v = 0u;
            if (ok) v = __ldg(reinterpret_cast<const uint32_t *>(table + (int64_t)id * row_bytes) + piece);
            reinterpret_cast<uint32_t *>(out)[g] = v;
        }
    }
}

// ---- int32 -> int64 -------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) widen_kernel(const int32_t *in, int64_t n, int64_t *out) {
    const bool vec = ((reinterpret_cast<uintptr_t>(in) & 15) == 0) && ((reinterpret_cast<uintptr_t>(out) & 15) == 0);
    const int64_t n4 = vec ? n >> 2 : 0;
    for (int64_t g = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; g < n4; g += (int64_t)gridDim.x * blockDim.x) {
        const int4 v = __ldg(reinterpret_cast<const int4 *>(in) + g);
        reinterpret_cast<longlong2 *>(out)[2 * g] = make_longlong2(v.x, v.y);
        reinterpret_cast<longlong2 *>(out)[2 * g + 1] = make_longlong2(v.z, v.w);
    }
    for (int64_t i = 4 * n4 + (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x)
        out[i] = in[i];
}

}  // namespace dtk
