// dnatok_api.cu -- host side of the C-ABI declared in include/dnatok.h.
//
// Argument marshalling, scratch management and the pinned multi-stream scheduler; every
// step of the hot path itself runs in the kernels of encode_v5.cuh / encode_v7.cuh / bpe_kernel.cuh /
// pad_kernel.cuh.  There is no CPU fallback anywhere in this file.
#include "../../include/dnatok.h"

#include <algorithm>
#include <cstdarg>
#include <cstdint>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <string>
#include <vector>

#include "bpe_kernel.cuh"
#include "common.cuh"
#include "encode_v5.cuh"
#include "encode_v7.cuh"
#include "encode_fasta.cuh"
#include "ext_kernels.cuh"
#include "pad_kernel.cuh"

using namespace dtk;

// ---- dnatok_decode_static's scratch: decoded bytes per record, DNATOK_DECODE_STATIC_MAX_RECORDS x int32 = 4 MiB, held by
// every GPU that loads the library until the process exits.  In host code this name is a host-side stand-in, not a device
// address: the device address of the array on a given GPU comes from cudaGetSymbolAddress with that GPU current
// (static_scratch_on below), once per device, and is what the kernels are given.
static __device__ __align__(256) int32_t g_decode_static_rec_len[DNATOK_DECODE_STATIC_MAX_RECORDS];

namespace {

// device address of g_decode_static_rec_len on `device`, which must be the current device; resolved once per device
int32_t *static_scratch_on(int device) {
    constexpr int MAX_DEV = 64;
    static std::mutex mu;
    static int32_t *addr[MAX_DEV] = {};
    if (device < 0 || device >= MAX_DEV) return nullptr;
    std::lock_guard<std::mutex> lock(mu);
    if (!addr[device]) {
        void *ptr = nullptr;
        if (cudaGetSymbolAddress(&ptr, g_decode_static_rec_len) != cudaSuccess || !ptr) { cudaGetLastError(); return nullptr; }
        addr[device] = static_cast<int32_t *>(ptr);
    }
    return addr[device];
}

// scan scratch of one in-flight encode: tile descriptors, ticket counter, host-mapped status words
struct EncCtx {
    TileDesc *descs = nullptr;
    TileDesc *gdescs = nullptr;        // [descs_cap / 32 + 2] group aggregates of the two-level look-back
    uint32_t *ls = nullptr;            // [descs_cap] line-state chain words
    int64_t *first_rec = nullptr;      // [descs_cap + 1] record range of every super-tile (pre-pass output)
    int64_t descs_cap = 0;
    int32_t *rec_k = nullptr;          // [reck_cap] kept-base index of every record start (many-starts path)
    int64_t reck_cap = 0;
    unsigned long long *ticket = nullptr;
    unsigned long long ticket_base = 0;
    uint32_t *h_status = nullptr;      // pinned + mapped: [0] capacity overflow, [1] scan protocol failure, [2] a layout check failed
    int fa_skip = 0;                   // calls left that go to the chained-scan encoder directly after a failed layout check
    uint32_t *d_status = nullptr;      // device alias of h_status
    uint32_t gen = 0;
    unsigned long long *prof = nullptr;   // phase timers of debug builds (-DDTK_PROF)
    // regular-layout fast path (encode_fasta.cuh)
    int32_t *fa_par = nullptr, *fa_tok = nullptr; int64_t fa_rec_cap = 0;
    int32_t *fa_first = nullptr; int64_t fa_tile_cap = 0;
    uint32_t *fa_flag = nullptr;
    bool fa_tried = false;             // the last strip-path call on this context went through the regular-layout encoder
    // BPE pass scratch
    uint8_t *cls = nullptr;  int64_t cls_cap = 0;
    uint16_t *tmp_tok = nullptr;
    int64_t *koff = nullptr; int32_t *tok_cnt = nullptr; int64_t rec_cap = 0;
    BpeSeg *segs = nullptr; int64_t segs_cap = 0;   // bin-sorted ACGT segments of 2 or more symbols
    uint32_t *bpe_ctl = nullptr;                    // bin counts, list slots, work items, work-item counters
    uint32_t *bpe_hist = nullptr; int64_t bpe_hist_cap = 0;   // per-CTA bin counts of the segment finder
};

struct StreamSlot {
    uint8_t *d_buf = nullptr;
    int64_t *d_recoff = nullptr, *h_recoff = nullptr;
    void *d_ids = nullptr;
    int64_t *d_out_off = nullptr;
    int32_t *d_batch = nullptr;
    uint8_t *d_mask = nullptr;
    cudaEvent_t ev_h2d = nullptr, ev_carry = nullptr, ev_done = nullptr, ev_off = nullptr;
    EncCtx ctx;
};

struct StreamRing {
    int64_t chunk_bytes = 0, carry_cap = 0, max_rows = 0;
    int n_streams = 0, n_slots = 0;
    std::vector<cudaStream_t> streams;
    std::vector<StreamSlot> slots;
    // pinned staging ring for a producer that reads from a file or from pageable memory: n_streams + 1 slots of chunk_bytes
    std::vector<uint8_t *> stage;
    std::vector<cudaEvent_t> ev_stage;           // the H2D copy out of the slot has finished
};

}  // namespace

struct dnatok {
    dnatok_config cfg;
    int device = 0;
    int sm_count = 0;
    EncParams prm;
    uint8_t *d_lut = nullptr;
    uint64_t *d_table = nullptr;
    int32_t *d_kmer_lut = nullptr, *d_remap4 = nullptr;   // table-driven k-mer ids (nullptr: base-4 closed form)
    uint32_t *d_spell_off = nullptr;   // BPE decode: [4 + n_merges + 1] offsets of the token spellings
    uint8_t *d_spell = nullptr;        //             the spellings, back to back (nullptr: too long to keep, decode unavailable)
    int32_t *d_rec_len = nullptr; int64_t rec_len_cap = 0;   // decode: decoded bytes per record
    int32_t *d_static_rec_len = nullptr;                     // decode_static: device address of g_decode_static_rec_len on h->device
    uint32_t table_mask = 0;
    int32_t bpe_cap = 0;
    EncCtx ctx;
    StreamRing ring;
    int enc_ctas_per_sm = 1, dense_ctas_per_sm = 1, bpe_ctas_per_sm = 1;
    bool dense = false;                // no SKIP class and strip_headers == 0: kept bases = bytes, the no-scan encoder runs
    int force_S = 0;                   // dnatok_set_super_tile: fixed super-tile size in sub-tiles (0 = automatic)
    int fast_path = 1;                 // dnatok_set_fast_path: 1 = try the regular-layout encoder first on inputs of 48 MiB or more,
                                       //   2 = on every input, 0 = chained-scan encoder only
    int fasta_ctas_per_sm = 4;
    int grid_cap = 0;                  // dnatok_set_grid_cap: at most this many persistent CTAs per launch (0 = no cap)
    int64_t launches = 0;
    std::string err;
};

namespace {

int fail(dnatok_t *h, int code, const char *fmt, ...) {
    if (h) {
        char buf[512];
        va_list ap; va_start(ap, fmt); vsnprintf(buf, sizeof buf, fmt, ap); va_end(ap);
        h->err = buf;
    }
    return code;
}

// selects the handle's device for the duration of an entry point and gives the caller's device back afterwards
struct DeviceGuard {
    int prev = -1, cur = -1;
    bool ok = false;
    explicit DeviceGuard(int d) : cur(d) { ok = cudaGetDevice(&prev) == cudaSuccess && (prev == d || cudaSetDevice(d) == cudaSuccess); }
    ~DeviceGuard() { if (prev >= 0 && prev != cur) cudaSetDevice(prev); }
    DeviceGuard(const DeviceGuard &) = delete;
    DeviceGuard &operator=(const DeviceGuard &) = delete;
};
#define USE_DEVICE(h) DeviceGuard dev_guard_((h)->device); if (!dev_guard_.ok) return fail((h), DNATOK_ECUDA, "cannot select device %d", (h)->device)

#define CU(call)                                                                                      \
    do {                                                                                              \
        cudaError_t e_ = (call);                                                                      \
        if (e_ != cudaSuccess)                                                                        \
            return fail(h, e_ == cudaErrorMemoryAllocation ? DNATOK_ENOMEM : DNATOK_ECUDA, "%s: %s", \
                        #call, cudaGetErrorString(e_));                                               \
    } while (0)

void default_lut(uint8_t *lut) {
    for (int b = 0; b < 256; ++b) lut[b] = DNATOK_CLS_UNK;
    const char *up = "ACGTN", *lo = "acgtn";
    for (int i = 0; i < 5; ++i) { lut[(uint8_t)up[i]] = (uint8_t)i; lut[(uint8_t)lo[i]] = (uint8_t)i; }
    lut['\n'] = DNATOK_CLS_SKIP; lut['\r'] = DNATOK_CLS_SKIP;
}

uint32_t host_hash(uint32_t key) {   // must match bpe_hash()
    key ^= key >> 15; key *= 0x2c1b3c6du; key ^= key >> 12; key *= 0x297a2d39u; key ^= key >> 15;
    return key;
}

int ctx_init(dnatok_t *h, EncCtx &c) {
    CU(cudaMalloc(&c.ticket, sizeof(unsigned long long)));
    CU(cudaMemset(c.ticket, 0, sizeof(unsigned long long)));
    CU(cudaHostAlloc(&c.h_status, 4 * sizeof(uint32_t), cudaHostAllocMapped));
    c.h_status[0] = c.h_status[1] = c.h_status[2] = c.h_status[3] = 0;
    CU(cudaHostGetDevicePointer((void **)&c.d_status, c.h_status, 0));
    CU(cudaMalloc(&c.prof, 64 * sizeof(unsigned long long)));
    CU(cudaMemset(c.prof, 0, 64 * sizeof(unsigned long long)));
    return DNATOK_OK;
}

void ctx_free(EncCtx &c) {
    cudaFree(c.descs); cudaFree(c.gdescs); cudaFree(c.ls); cudaFree(c.first_rec); cudaFree(c.rec_k); cudaFree(c.ticket); cudaFreeHost(c.h_status);
    cudaFree(c.prof);
    cudaFree(c.fa_par); cudaFree(c.fa_tok); cudaFree(c.fa_first); cudaFree(c.fa_flag);
    cudaFree(c.cls); cudaFree(c.tmp_tok); cudaFree(c.koff); cudaFree(c.tok_cnt); cudaFree(c.segs); cudaFree(c.bpe_ctl); cudaFree(c.bpe_hist);
    c = EncCtx();
}

// stream-ordered growth of the tile-descriptor array (never synchronises the host)
int ctx_reserve_tiles(dnatok_t *h, EncCtx &c, int64_t n_tiles, int64_t n_rec, cudaStream_t st) {
    if (n_rec + 1 > c.reck_cap) {
        int64_t cap = std::max<int64_t>(n_rec + 1 + n_rec / 4, 1024);
        if (c.rec_k) CU(cudaFreeAsync(c.rec_k, st));
        c.rec_k = nullptr; c.reck_cap = 0;
        CU(cudaMallocAsync((void **)&c.rec_k, (size_t)cap * sizeof(int32_t), st));
        c.reck_cap = cap;
    }
    if (n_tiles <= c.descs_cap) return DNATOK_OK;
    int64_t cap = std::max<int64_t>(n_tiles + n_tiles / 4, 1024);
    if (c.descs) CU(cudaFreeAsync(c.descs, st));
    if (c.gdescs) CU(cudaFreeAsync(c.gdescs, st));
    if (c.ls) CU(cudaFreeAsync(c.ls, st));
    if (c.first_rec) CU(cudaFreeAsync(c.first_rec, st));
    c.descs = nullptr; c.gdescs = nullptr; c.ls = nullptr; c.first_rec = nullptr; c.descs_cap = 0;
    CU(cudaMallocAsync((void **)&c.descs, (size_t)cap * sizeof(TileDesc), st));
    CU(cudaMallocAsync((void **)&c.gdescs, (size_t)(cap / 32 + 2) * sizeof(TileDesc), st));
    CU(cudaMemsetAsync(c.gdescs, 0, (size_t)(cap / 32 + 2) * sizeof(TileDesc), st));
    CU(cudaMallocAsync((void **)&c.ls, (size_t)cap * sizeof(uint32_t), st));
    CU(cudaMallocAsync((void **)&c.first_rec, (size_t)(cap + 1) * sizeof(int64_t), st));
    CU(cudaMemsetAsync(c.descs, 0, (size_t)cap * sizeof(TileDesc), st));
    CU(cudaMemsetAsync(c.ls, 0, (size_t)cap * sizeof(uint32_t), st));
    c.descs_cap = cap;
    return DNATOK_OK;
}

int ctx_reserve_fasta(dnatok_t *h, EncCtx &c, int64_t n_rec, int64_t n_wtiles, cudaStream_t st) {
    if (!c.fa_flag) CU(cudaMallocAsync((void **)&c.fa_flag, 16, st));
    if (n_rec + 1 > c.fa_rec_cap) {
        if (c.fa_par) CU(cudaFreeAsync(c.fa_par, st));
        if (c.fa_tok) CU(cudaFreeAsync(c.fa_tok, st));
        c.fa_par = nullptr; c.fa_tok = nullptr; c.fa_rec_cap = 0;
        const int64_t cap = n_rec + n_rec / 4 + 1024;
        CU(cudaMallocAsync((void **)&c.fa_par, (size_t)cap * 4 * sizeof(int32_t), st));
        CU(cudaMallocAsync((void **)&c.fa_tok, (size_t)cap * sizeof(int32_t), st));
        c.fa_rec_cap = cap;
    }
    if (n_wtiles + 1 > c.fa_tile_cap) {
        if (c.fa_first) CU(cudaFreeAsync(c.fa_first, st));
        c.fa_first = nullptr; c.fa_tile_cap = 0;
        const int64_t cap = n_wtiles + n_wtiles / 4 + 1024;
        CU(cudaMallocAsync((void **)&c.fa_first, (size_t)cap * sizeof(int32_t), st));
        c.fa_tile_cap = cap;
    }
    return DNATOK_OK;
}

int ctx_next_gen(dnatok_t *h, EncCtx &c, cudaStream_t st) {
    if (++c.gen >= (1u << 24) - 1) {       // generation tags are 24 bits wide in TileDesc::l_word
        if (c.descs) CU(cudaMemsetAsync(c.descs, 0, (size_t)c.descs_cap * sizeof(TileDesc), st));
        if (c.gdescs) CU(cudaMemsetAsync(c.gdescs, 0, (size_t)(c.descs_cap / 32 + 2) * sizeof(TileDesc), st));
        if (c.ls) CU(cudaMemsetAsync(c.ls, 0, (size_t)c.descs_cap * sizeof(uint32_t), st));
        c.gen = 1;
    }
    return DNATOK_OK;
}

// launch of an encode kernel behind its pre-pass with programmatic stream serialisation (the kernel's prologue overlaps
// the pre-pass's tail; the kernel waits with griddepcontrol.wait before it reads what the pre-pass wrote)
template <typename K>
void launch_pdl(K kernel, int grid, int block, size_t smem, cudaStream_t st, const EncArgs &a, bool pdl) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)grid); cfg.blockDim = dim3((unsigned)block); cfg.dynamicSmemBytes = smem; cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr; cfg.numAttrs = pdl ? 1 : 0;
    cudaLaunchKernelEx(&cfg, kernel, a);
}

// the headline shapes get a kernel with only their own emission variant compiled in (smaller instruction footprint)
template <typename IdT>
void launch_dense(const EncArgs &a, int kk, int grid, cudaStream_t st) {
    constexpr bool wide = sizeof(IdT) >= 2;                    // uint8 ids: the BPE class pass, single-nt only
    switch (wide ? kk : 0) {
        case 0: launch_pdl(v7::encode_tiles_v7<IdT, 0, true>, grid, v7::NT7, sizeof(v7::Smem7), st, a, true); break;
        case 1: launch_pdl(v7::encode_tiles_v7<IdT, wide ? 1 : 0, true>, grid, v7::NT7, sizeof(v7::Smem7), st, a, true); break;
        case 2: launch_pdl(v7::encode_tiles_v7<IdT, wide ? 2 : 0, true>, grid, v7::NT7, sizeof(v7::Smem7), st, a, true); break;
        case 3: launch_pdl(v7::encode_tiles_v7<IdT, wide ? 3 : 0, true>, grid, v7::NT7, sizeof(v7::Smem7), st, a, true); break;
        case 4: launch_pdl(v7::encode_tiles_v7<IdT, wide ? 4 : 0, true>, grid, v7::NT7, sizeof(v7::Smem7), st, a, true); break;
        case 5: launch_pdl(v7::encode_tiles_v7<IdT, wide ? 5 : 0, true>, grid, v7::NT7, sizeof(v7::Smem7), st, a, true); break;
        case 6: launch_pdl(v7::encode_tiles_v7<IdT, wide ? 6 : 0, true>, grid, v7::NT7, sizeof(v7::Smem7), st, a, true); break;
        case 8: launch_pdl(v7::encode_tiles_v7<IdT, wide ? 8 : 0, true>, grid, v7::NT7, sizeof(v7::Smem7), st, a, true); break;
        default: launch_pdl(v7::encode_tiles_v7<IdT, wide ? -1 : 0, true>, grid, v7::NT7, sizeof(v7::Smem7), st, a, true); break;
    }
}
template <typename K, typename... Args>
void launch_pdl1(K kernel, int grid, int block, size_t smem, cudaStream_t st, bool pdl, Args... args) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)grid); cfg.blockDim = dim3((unsigned)block); cfg.dynamicSmemBytes = smem; cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr; cfg.numAttrs = pdl ? 1 : 0;
    cudaLaunchKernelEx(&cfg, kernel, args...);
}
// The regular-layout path costs three launches and a latency-bound parse before its encoder starts; measured against the
// chained-scan encoder on L2-flushed inputs of both FASTA shapes it wins from 32-64 MiB on.
constexpr int64_t FAST_PATH_MIN_BYTES = 48ll << 20;
constexpr int FAST_PATH_SKIP_CALLS = 8;

template <typename IdT, bool FUSED = false>
void launch_fasta(const fa::FastaArgs &f, int kk, int grid, cudaStream_t st) {
    using namespace dtk::fa;
    constexpr bool wide = sizeof(IdT) >= 2;
    const size_t sm = sizeof(SmemFa);
    switch (wide ? kk : 0) {
        case 0: launch_pdl1(encode_fasta_kernel<IdT, 0, FUSED>, grid, FW_WARPS * 32, sm, st, true, f); break;
        case 1: launch_pdl1(encode_fasta_kernel<IdT, wide ? 1 : 0, FUSED>, grid, FW_WARPS * 32, sm, st, true, f); break;
        case 2: launch_pdl1(encode_fasta_kernel<IdT, wide ? 2 : 0, FUSED>, grid, FW_WARPS * 32, sm, st, true, f); break;
        case 3: launch_pdl1(encode_fasta_kernel<IdT, wide ? 3 : 0, FUSED>, grid, FW_WARPS * 32, sm, st, true, f); break;
        case 4: launch_pdl1(encode_fasta_kernel<IdT, wide ? 4 : 0, FUSED>, grid, FW_WARPS * 32, sm, st, true, f); break;
        case 5: launch_pdl1(encode_fasta_kernel<IdT, wide ? 5 : 0, FUSED>, grid, FW_WARPS * 32, sm, st, true, f); break;
        case 6: launch_pdl1(encode_fasta_kernel<IdT, wide ? 6 : 0, FUSED>, grid, FW_WARPS * 32, sm, st, true, f); break;
        case 8: launch_pdl1(encode_fasta_kernel<IdT, wide ? 8 : 0, FUSED>, grid, FW_WARPS * 32, sm, st, true, f); break;
        default: launch_pdl1(encode_fasta_kernel<IdT, wide ? -1 : 0, FUSED>, grid, FW_WARPS * 32, sm, st, true, f); break;
    }
}
template <typename IdT>
void launch_strip(const EncArgs &a, int kk, int grid, cudaStream_t st, bool chained) {
    using namespace dtk::v5;
    constexpr bool wide = sizeof(IdT) >= 2;
    switch (wide ? kk : 0) {
        case 0: launch_pdl(encode_tiles_v5<IdT, 0>, grid, NT, sizeof(Smem5), st, a, a.first_rec != nullptr || chained); break;
        case 1: launch_pdl(encode_tiles_v5<IdT, wide ? 1 : 0>, grid, NT, sizeof(Smem5), st, a, a.first_rec != nullptr || chained); break;
        case 2: launch_pdl(encode_tiles_v5<IdT, wide ? 2 : 0>, grid, NT, sizeof(Smem5), st, a, a.first_rec != nullptr || chained); break;
        case 3: launch_pdl(encode_tiles_v5<IdT, wide ? 3 : 0>, grid, NT, sizeof(Smem5), st, a, a.first_rec != nullptr || chained); break;
        case 4: launch_pdl(encode_tiles_v5<IdT, wide ? 4 : 0>, grid, NT, sizeof(Smem5), st, a, a.first_rec != nullptr || chained); break;
        case 5: launch_pdl(encode_tiles_v5<IdT, wide ? 5 : 0>, grid, NT, sizeof(Smem5), st, a, a.first_rec != nullptr || chained); break;
        case 6: launch_pdl(encode_tiles_v5<IdT, wide ? 6 : 0>, grid, NT, sizeof(Smem5), st, a, a.first_rec != nullptr || chained); break;
        case 8: launch_pdl(encode_tiles_v5<IdT, wide ? 8 : 0>, grid, NT, sizeof(Smem5), st, a, a.first_rec != nullptr || chained); break;
        default: launch_pdl(encode_tiles_v5<IdT, wide ? -1 : 0>, grid, NT, sizeof(Smem5), st, a, a.first_rec != nullptr || chained); break;
    }
}

int pad_on(dnatok_t *h, const void *d_ids, const int64_t *d_out_off, int64_t n_rec, int32_t *d_batch,
           uint8_t *d_mask, cudaStream_t st, int64_t ids_cap, const uint32_t *run_if);

// d_batch != nullptr asks for the padded batch as well (handle with seq_len > 0).  If the regular-layout encoder takes the call
// it writes the tokens straight into the batch (*fused = true: batch and mask are complete when the launches below have run,
// whichever encoder ends up serving the call); otherwise *fused stays false and the caller runs the pad kernel on the ids.
template <typename IdT>
int launch_tiles(dnatok_t *h, EncCtx &c, const EncParams &prm, const uint8_t *d_bytes, int64_t n_bytes,
                 const int64_t *d_rec_off, int64_t n_rec, int64_t off_bias, void *ids, int64_t ids_cap,
                 int64_t *out_off, cudaStream_t st, int32_t *d_batch = nullptr, uint8_t *d_mask = nullptr,
                 bool *fused = nullptr) {
    EncArgs a;
    uintptr_t addr = reinterpret_cast<uintptr_t>(d_bytes);
    a.mis = (int64_t)(addr & 15);
    a.bytes_al = reinterpret_cast<const uint8_t *>(addr - (uintptr_t)a.mis);
    a.p_end = a.mis + n_bytes;
    // tile size: large inputs want large tiles (the per-tile scan work is amortised over S x 16 KiB); small inputs
    // want enough tiles to occupy every CTA slot a few times over; the no-scan encoder also wants few record starts
    // per tile (its segment tables hold v7::EV_MAX)
    const bool dense = h->dense;
    const int64_t slots = (int64_t)h->sm_count * (dense ? h->dense_ctas_per_sm : h->enc_ctas_per_sm);
    int S = S_MAX;
    while (S > 1 && a.p_end / ((int64_t)S * TB) + 1 < 3 * slots) S >>= 1;
    while (dense && S > 1 && n_rec * (int64_t)S * TB > (v7::EV_MAX / 2) * std::max<int64_t>(n_bytes, 1)) S >>= 1;
    if (h->force_S > 0) S = h->force_S;
    a.S = S;
    int64_t n_tiles = a.p_end / ((int64_t)S * TB) + 1;
    if (n_tiles > 0x7fffffff) return fail(h, DNATOK_EINVAL, "n_bytes too large for one call");
    const int64_t n_scan_blocks = dense ? (n_rec + v7::DS_BLK - 1) / v7::DS_BLK + (n_rec == 0) : 0;
    int rc = ctx_reserve_tiles(h, c, std::max(n_tiles, n_scan_blocks), n_rec, st); if (rc) return rc;
    rc = ctx_next_gen(h, c, st); if (rc) return rc;
    a.rec_off = d_rec_off; a.n_rec = n_rec; a.off_bias = off_bias;
    a.ids = ids; a.ids_cap = ids_cap; a.out_off = out_off; a.out_bias = 0;
    a.lut = h->d_lut; a.descs = c.descs; a.gdescs = c.gdescs; a.ls = c.ls; a.rec_k = c.rec_k; a.first_rec = c.first_rec; a.ticket = c.ticket; a.ticket_base = c.ticket_base;
    a.status = c.d_status; a.prof = c.prof; a.gen = c.gen; a.n_tiles = (int32_t)n_tiles; a.prm = prm;
    a.run_if = nullptr;
    int grid = (int)std::min<int64_t>(n_tiles, slots);
    if (h->grid_cap > 0) grid = std::min(grid, h->grid_cap);
    // table-driven ids are compiled into the run-time-switch variant only (the per-k variants stay lean)
    const int kk = prm.mode == MODE_KMER ? (prm.remap4 ? 99 : prm.k) : 0;
    const unsigned nb_first = (unsigned)((n_tiles + 1 + 255) / 256);
    if (dense) {
        // record range of every tile + out_offsets (closed form from the record lengths), one launch
        v7::dense_prepass_kernel<<<nb_first + (unsigned)n_scan_blocks, v7::DS_NT, 0, st>>>(a, c.descs, (int)nb_first);
        CU(cudaGetLastError());
        h->launches += 1;
        launch_dense<IdT>(a, kk, grid, st);
    } else {
        bool chained = false;                                 // the kernels below follow kernels of this call
        bool f_fused = false;
        c.fa_tried = false;
        // (many short records: more than FW_MAXSEG of them would meet in some 16 KiB tile and fail the layout check anyway,
        // so an input that averages over half of that goes to the chained-scan encoder directly)
        const bool short_recs = h->fast_path != 2 && n_rec > (n_bytes / fa::FW_TILE + 1) * (fa::FW_MAXSEG / 2);
        // A failed layout check costs the regular-layout encoder's time on top of the chained scan's.  Inputs of one source tend
        // to be alike, so after a failure (reported by the fall-back launch through a host-mapped word; read here without any
        // synchronisation, so it may be seen a call or two late) the next FAST_PATH_SKIP_CALLS calls on this context skip the attempt.
        if (((volatile uint32_t *)c.h_status)[2]) { c.h_status[2] = 0; c.fa_skip = FAST_PATH_SKIP_CALLS; }
        bool try_fast = (h->fast_path == 2 || (h->fast_path == 1 && n_bytes >= FAST_PATH_MIN_BYTES)) && n_rec < (1ll << 31) && !short_recs;
        if (try_fast && h->fast_path == 1 && c.fa_skip > 0) { --c.fa_skip; try_fast = false; }
        if (try_fast) {
            // regular-layout fast path first (encode_fasta.cuh); the chained-scan encoder behind it runs only if the layout
            // check failed somewhere
            const int64_t n_wtiles = (a.p_end + fa::FW_TILE - 1) / fa::FW_TILE;
            const int64_t nb_scan = std::max<int64_t>(1, (n_rec + fa::OS_BLK - 1) / fa::OS_BLK);
            rc = ctx_reserve_tiles(h, c, std::max(n_tiles, nb_scan), n_rec, st); if (rc) return rc;
            rc = ctx_reserve_fasta(h, c, n_rec, n_wtiles, st); if (rc) return rc;
            a.descs = c.descs; a.gdescs = c.gdescs; a.ls = c.ls; a.rec_k = c.rec_k; a.first_rec = c.first_rec;
            CU(cudaMemsetAsync(c.fa_flag, 0, 16, st));
            fa::FastaArgs f;
            f.e = a; f.par = c.fa_par; f.rec_tok = c.fa_tok; f.wt_first = c.fa_first; f.irregular = c.fa_flag;
            f.n_wtiles = (int32_t)n_wtiles;
            const bool fuse = d_batch != nullptr && fused != nullptr && n_rec > 0 && sizeof(IdT) >= 2;
            f.seq_len = 0; f.pad_side = 0;
            if (fuse) {
                f.seq_len = h->cfg.seq_len; f.pad_side = h->cfg.pad_side;
                f.e.ids = d_batch; f.e.ids_cap = n_rec * (int64_t)h->cfg.seq_len;
            }
            const int64_t nthr = n_rec + n_wtiles;                       // one thread per tile, then one per record
            fa::fasta_parse_kernel<<<(unsigned)std::max<int64_t>(1, (nthr + 255) / 256), 256, 0, st>>>(f);
            launch_pdl1(fa::offsets_scan_kernel, (int)nb_scan, fa::OS_NT, 0, st, true, (const int32_t *)c.fa_tok, n_rec, out_off, (int64_t)0, c.descs, a.gen, c.d_status);
            int fgrid = (int)std::min<int64_t>((n_wtiles + fa::FW_WARPS - 1) / fa::FW_WARPS, (int64_t)h->sm_count * h->fasta_ctas_per_sm);
            fgrid = std::max(fgrid, 1);
            if (h->grid_cap > 0) fgrid = std::min(fgrid, h->grid_cap);
            if (fuse) {
                fa::PadFillArgs pf;
                pf.out_off = out_off; pf.n_rows = n_rec; pf.batch_ids = d_batch; pf.mask = d_mask;
                pf.seq_len = h->cfg.seq_len; pf.pad_side = h->cfg.pad_side; pf.pad_id = h->cfg.pad_id;
                int pgrid = (int)std::min<int64_t>(n_rec, (int64_t)h->sm_count * 16);
                if (h->grid_cap > 0) pgrid = std::min(pgrid, h->grid_cap);
                launch_pdl1(fa::pad_fill_kernel, pgrid, 256, 0, st, true, pf);
                launch_fasta<int32_t, true>(f, kk, fgrid, st);           // the batch holds int32 whatever the id type
                h->launches += 1;
            } else launch_fasta<IdT>(f, kk, fgrid, st);
            CU(cudaGetLastError());
            h->launches += 3;
            rc = ctx_next_gen(h, c, st); if (rc) return rc;      // the scan above used this generation's chain words
            a.gen = c.gen; a.run_if = c.fa_flag;
            chained = true;
            f_fused = fuse;
            c.fa_tried = true;
        }
        // an input that gives every CTA at most one tile is encoded in ONE launch: the record range of a tile is searched
        // inside the kernel instead of by the pre-pass (SURVEY.md section 7 hard part 6)
        if (n_tiles <= slots && n_rec <= (1 << 16)) a.first_rec = nullptr;
        else {
            launch_pdl1(v5::tile_first_rec_kernel, (int)nb_first, 256, 0, st, chained, a);
            CU(cudaGetLastError());
            h->launches += 1;
        }
        launch_strip<IdT>(a, kk, grid, st, chained);
        if (chained && f_fused) {
            // the chained-scan encoder's ids go through the pad kernel, which like it returns at once unless the flag is set
            CU(cudaGetLastError());
            rc = pad_on(h, ids, out_off, n_rec, d_batch, d_mask, st, ids_cap, c.fa_flag); if (rc) return rc;
            *fused = true;
        }
    }
    CU(cudaGetLastError());
    c.ticket_base += (unsigned long long)n_tiles + (unsigned long long)grid;
    h->launches += 1;
    return DNATOK_OK;
}

int ctx_reserve_bpe(dnatok_t *h, EncCtx &c, int64_t n_bytes, int64_t n_rec, cudaStream_t st) {
    if (n_bytes > c.cls_cap) {
        int64_t cap = n_bytes + n_bytes / 8 + 256;
        if (c.cls) CU(cudaFreeAsync(c.cls, st));
        if (c.tmp_tok) CU(cudaFreeAsync(c.tmp_tok, st));
        c.cls = nullptr; c.tmp_tok = nullptr; c.cls_cap = 0;
        CU(cudaMallocAsync((void **)&c.cls, (size_t)cap, st));
        CU(cudaMallocAsync((void **)&c.tmp_tok, (size_t)cap * sizeof(uint16_t), st));
        c.cls_cap = cap;
    }
    if (!c.bpe_ctl) CU(cudaMallocAsync((void **)&c.bpe_ctl, CTL_WORDS * sizeof(uint32_t), st));
    if (n_rec + 1 > c.rec_cap) {
        int64_t cap = n_rec + n_rec / 8 + 256;
        if (c.koff) CU(cudaFreeAsync(c.koff, st));
        if (c.tok_cnt) CU(cudaFreeAsync(c.tok_cnt, st));
        c.koff = nullptr; c.tok_cnt = nullptr; c.rec_cap = 0;
        CU(cudaMallocAsync((void **)&c.koff, (size_t)cap * sizeof(int64_t), st));
        CU(cudaMallocAsync((void **)&c.tok_cnt, (size_t)cap * sizeof(int32_t), st));
        c.rec_cap = cap;
    }
    return DNATOK_OK;
}


int encode_on(dnatok_t *h, EncCtx &c, const uint8_t *d_bytes, int64_t n_bytes, const int64_t *d_rec_off,
              int64_t n_rec, int64_t off_bias, void *d_ids, int64_t ids_cap, int64_t *d_out_off, cudaStream_t st,
              int32_t *d_batch = nullptr, uint8_t *d_mask = nullptr, bool *fused = nullptr) {
    const dnatok_config &cfg = h->cfg;
    if (cfg.mode != DNATOK_BPE) {
        if (cfg.id_dtype == DNATOK_I16)
            return launch_tiles<int16_t>(h, c, h->prm, d_bytes, n_bytes, d_rec_off, n_rec, off_bias, d_ids, ids_cap, d_out_off, st,
                                         d_batch, d_mask, fused);
        return launch_tiles<int32_t>(h, c, h->prm, d_bytes, n_bytes, d_rec_off, n_rec, off_bias, d_ids, ids_cap, d_out_off, st,
                                     d_batch, d_mask, fused);
    }
    // BPE: pass A = compact kept classes + kept-base CSR offsets (the single-nt encoder with class ids),
    //      pass B = merge kernel per read, pass C = offsets scan, pass D = gather into ids_out
    int rc = ctx_reserve_bpe(h, c, n_bytes, n_rec, st); if (rc) return rc;
    EncParams pa = h->prm;
    pa.mode = MODE_SINGLE_NT; pa.k = 1; pa.unk_id = DNATOK_CLS_UNK;
    for (int i = 0; i < 5; ++i) pa.nt_ids[i] = i;
    rc = launch_tiles<uint8_t>(h, c, pa, d_bytes, n_bytes, d_rec_off, n_rec, off_bias, c.cls, c.cls_cap, c.koff, st);
    if (rc) return rc;
    if (n_rec > 0) {
        if (n_bytes >= (1ll << 32)) return fail(h, DNATOK_EINVAL, "BPE: one call encodes less than 4 GiB (split the input)");
        // a segment of two or more symbols is followed by a boundary symbol or by the end of its read
        if (c.segs_cap < n_bytes / 3 + n_rec + 16) {
            if (c.segs) CU(cudaFreeAsync(c.segs, st));
            c.segs = nullptr; c.segs_cap = 0;
            const int64_t scap = n_bytes / 3 + n_rec + n_rec / 8 + 16;
            CU(cudaMallocAsync((void **)&c.segs, (size_t)scap * sizeof(BpeSeg), st));
            c.segs_cap = scap;
        }
        const unsigned nb_seg = (unsigned)((n_rec + BPE_SEG_WARPS - 1) / BPE_SEG_WARPS);
        if (c.bpe_hist_cap < (int64_t)nb_seg) {
            if (c.bpe_hist) CU(cudaFreeAsync(c.bpe_hist, st));
            c.bpe_hist = nullptr; c.bpe_hist_cap = 0;
            const int64_t hcap = (int64_t)nb_seg + nb_seg / 4 + 16;
            CU(cudaMallocAsync((void **)&c.bpe_hist, (size_t)hcap * BPE_NB * sizeof(uint32_t), st));
            c.bpe_hist_cap = hcap;
        }
        BpeArgs b;
        b.cta_hist = c.bpe_hist;
        b.cls = c.cls; b.koff = c.koff; b.n_rec = n_rec; b.table = h->d_table; b.table_mask = h->table_mask;
        b.tmp_tok = c.tmp_tok; b.tok_cnt = c.tok_cnt; b.status = c.d_status;
        b.segs = c.segs; b.segs_cap = c.segs_cap; b.ctl = c.bpe_ctl; b.giant_cap = h->bpe_cap;
        CU(cudaMemsetAsync(c.bpe_ctl, 0, CTL_WORDS * sizeof(uint32_t), st));
        bpe_segments_kernel<false><<<nb_seg, BPE_SEG_WARPS * 32, 0, st>>>(b);
        bpe_bins_kernel<<<1, 128, 0, st>>>(b);
        bpe_segments_kernel<true><<<nb_seg, BPE_SEG_WARPS * 32, 0, st>>>(b);
        int grid = h->sm_count * h->bpe_ctas_per_sm;
        if (h->grid_cap > 0) grid = std::min(grid, h->grid_cap);
        bpe_merge_kernel<<<grid, BPE_WARPS * 32, BPE_WARPS * BPE_SLOT_WORDS * sizeof(uint32_t), st>>>(b);
        if (h->bpe_cap > BPE_SLOT_WORDS) {
            int gg = h->sm_count;
            if (h->grid_cap > 0) gg = std::min(gg, h->grid_cap);
            bpe_merge_giant_kernel<<<gg, 32, (size_t)h->bpe_cap * sizeof(uint32_t), st>>>(b);
            h->launches += 1;
        }
        CU(cudaGetLastError());
        h->launches += 4;
    }
    scan_counts_kernel<<<1, 1024, 0, st>>>(c.tok_cnt, n_rec, d_out_off);
    CU(cudaGetLastError());
    h->launches += 1;
    if (n_rec > 0) {
        int grid = (int)std::min<int64_t>((n_rec + 7) / 8, (int64_t)h->sm_count * 8);
        if (h->grid_cap > 0) grid = std::min(grid, h->grid_cap);
        if (cfg.id_dtype == DNATOK_I16)
            bpe_gather_kernel<int16_t><<<grid, 256, 0, st>>>(c.tmp_tok, c.koff, d_out_off, n_rec, (int16_t *)d_ids, ids_cap,
                                                           cfg.base_id, cfg.n_id, cfg.unk_id, c.d_status);
        else
            bpe_gather_kernel<int32_t><<<grid, 256, 0, st>>>(c.tmp_tok, c.koff, d_out_off, n_rec, (int32_t *)d_ids, ids_cap,
                                                           cfg.base_id, cfg.n_id, cfg.unk_id, c.d_status);
        CU(cudaGetLastError());
        h->launches += 1;
    }
    return DNATOK_OK;
}

int pad_on(dnatok_t *h, const void *d_ids, const int64_t *d_out_off, int64_t n_rec, int32_t *d_batch,
           uint8_t *d_mask, cudaStream_t st, int64_t ids_cap = INT64_MAX, const uint32_t *run_if = nullptr) {
    if (n_rec == 0) return DNATOK_OK;
    PadArgs a;
    a.run_if = run_if;
    a.ids = d_ids; a.out_off = d_out_off; a.n_rows = n_rec; a.batch_ids = d_batch; a.mask = d_mask;
    a.seq_len = h->cfg.seq_len; a.pad_side = h->cfg.pad_side; a.pad_id = h->cfg.pad_id;
    a.ids_cap = ids_cap;
    int grid = (int)std::min<int64_t>(n_rec, (int64_t)h->sm_count * 16);
    if (h->grid_cap > 0) grid = std::min(grid, h->grid_cap);
    if (h->cfg.id_dtype == DNATOK_I16) pad_rows_kernel<int16_t><<<grid, 256, 0, st>>>(a);
    else pad_rows_kernel<int32_t><<<grid, 256, 0, st>>>(a);
    CU(cudaGetLastError());
    h->launches += 1;
    return DNATOK_OK;
}

int status_of(dnatok_t *h, EncCtx &c) {
    int rc = DNATOK_OK;
    if (c.h_status[1]) rc = fail(h, DNATOK_ESTATE, "scan look-back spin limit hit (tile chain broken)");
    else if (c.h_status[0]) rc = fail(h, DNATOK_ECAPACITY, "an output buffer or workspace was too small");
    c.h_status[0] = c.h_status[1] = 0;
    return rc;
}

void ring_free(StreamRing &r) {
    for (auto &s : r.slots) {
        cudaFree(s.d_buf); cudaFree(s.d_recoff); cudaFreeHost(s.h_recoff); cudaFree(s.d_ids); cudaFree(s.d_out_off);
        cudaFree(s.d_batch); cudaFree(s.d_mask);
        if (s.ev_h2d) cudaEventDestroy(s.ev_h2d);
        if (s.ev_carry) cudaEventDestroy(s.ev_carry);
        if (s.ev_done) cudaEventDestroy(s.ev_done);
        if (s.ev_off) cudaEventDestroy(s.ev_off);
        ctx_free(s.ctx);
    }
    for (auto st : r.streams) cudaStreamDestroy(st);
    for (auto p : r.stage) cudaFreeHost(p);
    for (auto e : r.ev_stage) if (e) cudaEventDestroy(e);
    r = StreamRing();
}

int ring_setup(dnatok_t *h, int64_t chunk_bytes, int n_streams, int64_t max_rows) {
    StreamRing &r = h->ring;
    const int64_t carry_cap = (h->cfg.max_record_bytes + 255) & ~(int64_t)255;
    if (r.chunk_bytes == chunk_bytes && r.n_streams == n_streams && r.max_rows >= max_rows && r.carry_cap == carry_cap)
        return DNATOK_OK;
    ring_free(r);
    r.chunk_bytes = chunk_bytes; r.n_streams = n_streams; r.n_slots = std::max(2, n_streams);
    r.max_rows = max_rows; r.carry_cap = carry_cap;
    r.streams.resize(n_streams);
    for (auto &st : r.streams) CU(cudaStreamCreateWithFlags(&st, cudaStreamNonBlocking));
    r.slots.resize(r.n_slots);
    const int64_t cap = carry_cap + chunk_bytes;
    const size_t idsz = (size_t)h->cfg.id_dtype;
    for (auto &s : r.slots) {
        CU(cudaMalloc(&s.d_buf, (size_t)cap + 256));
        CU(cudaMalloc(&s.d_recoff, (size_t)(max_rows + 2) * sizeof(int64_t)));
        CU(cudaHostAlloc(&s.h_recoff, (size_t)(max_rows + 2) * sizeof(int64_t), cudaHostAllocDefault));
        CU(cudaMalloc(&s.d_ids, (size_t)cap * idsz));
        CU(cudaMalloc(&s.d_out_off, (size_t)(max_rows + 2) * sizeof(int64_t)));
        if (h->cfg.seq_len > 0) {
            CU(cudaMalloc(&s.d_batch, (size_t)max_rows * h->cfg.seq_len * sizeof(int32_t)));
            CU(cudaMalloc(&s.d_mask, (size_t)max_rows * h->cfg.seq_len));
        }
        CU(cudaEventCreateWithFlags(&s.ev_h2d, cudaEventDisableTiming));
        CU(cudaEventCreateWithFlags(&s.ev_carry, cudaEventDisableTiming));
        CU(cudaEventCreateWithFlags(&s.ev_done, cudaEventDisableTiming));
        CU(cudaEventCreateWithFlags(&s.ev_off, cudaEventDisableTiming));
        int rc = ctx_init(h, s.ctx); if (rc) return rc;
    }
    return DNATOK_OK;
}

int ring_stage_setup(dnatok_t *h) {
    StreamRing &r = h->ring;
    if (!r.stage.empty()) return DNATOK_OK;
    const int n = r.n_streams + 1;
    r.stage.assign(n, nullptr); r.ev_stage.assign(n, nullptr);
    for (int i = 0; i < n; ++i) {
        CU(cudaHostAlloc((void **)&r.stage[i], (size_t)r.chunk_bytes, cudaHostAllocDefault));
        CU(cudaEventCreateWithFlags(&r.ev_stage[i], cudaEventDisableTiming));
    }
    return DNATOK_OK;
}

}  // namespace

// ======================================================================================
extern "C" {

const char *dnatok_version(void) { return "dnatok-b200 0.1 (sm_100a)"; }

void dnatok_config_default(dnatok_config *cfg, int32_t mode, int32_t k) {
    memset(cfg, 0, sizeof *cfg);
    cfg->struct_size = sizeof *cfg;
    cfg->mode = mode; cfg->k = k; cfg->id_dtype = DNATOK_I32;
    default_lut(cfg->class_lut);
    cfg->strip_headers = 1; cfg->pad_id = 0; cfg->unk_id = 1;
    for (int i = 0; i < 5; ++i) cfg->nt_ids[i] = 2 + i;
    cfg->base_id = 3; cfg->n_id = 2; cfg->tail_policy = DNATOK_TAIL_PER_BASE;
    cfg->pad_side = DNATOK_PAD_LEFT; cfg->max_record_bytes = 1 << 20;
}

int dnatok_create(const dnatok_config *cfg_in, int device, dnatok_t **out) {
    if (!cfg_in || !out || cfg_in->struct_size != sizeof(dnatok_config)) return DNATOK_EINVAL;
    *out = nullptr;
    dnatok_config cfg = *cfg_in;
    bool zero = true;
    for (int b = 0; b < 256; ++b) zero = zero && cfg.class_lut[b] == 0;
    if (zero) default_lut(cfg.class_lut);
    for (int b = 0; b < 256; ++b)
        if (cfg.class_lut[b] > DNATOK_CLS_UNK && cfg.class_lut[b] != DNATOK_CLS_SKIP) return DNATOK_EINVAL;
    if (cfg.strip_headers && cfg.class_lut['\n'] != DNATOK_CLS_SKIP) return DNATOK_EINVAL;
    if (cfg.mode < DNATOK_SINGLE_NT || cfg.mode > DNATOK_BPE) return DNATOK_EINVAL;
    if (cfg.id_dtype != DNATOK_I16 && cfg.id_dtype != DNATOK_I32) return DNATOK_EINVAL;
    if (cfg.seq_len < 0 || (cfg.pad_side != DNATOK_PAD_LEFT && cfg.pad_side != DNATOK_PAD_RIGHT)) return DNATOK_EINVAL;
    if (cfg.max_record_bytes <= 0) cfg.max_record_bytes = 1 << 20;
    if (cfg.kmer_lut && cfg.mode != DNATOK_KMER) return DNATOK_EINVAL;
    int64_t max_id = std::max<int64_t>(cfg.unk_id, cfg.pad_id);
    if (cfg.mode == DNATOK_SINGLE_NT) {
        for (int i = 0; i < 5; ++i) max_id = std::max<int64_t>(max_id, cfg.nt_ids[i]);
    } else if (cfg.mode == DNATOK_KMER) {
        if (cfg.k < 1 || cfg.k > DNATOK_MAX_K) return DNATOK_EINVAL;
        if (cfg.tail_policy < DNATOK_TAIL_PER_BASE || cfg.tail_policy > DNATOK_TAIL_UNK) return DNATOK_EINVAL;
        int64_t fk = 1ll << (2 * cfg.k);
        max_id = std::max<int64_t>(max_id, cfg.base_id + fk - 1 + (cfg.tail_policy == DNATOK_TAIL_PER_BASE ? 5 : 0));
        if (max_id > 0x7fffffffll) return DNATOK_EINVAL;
        if (cfg.kmer_lut) {                                   // table-driven ids
            int64_t p5 = 1;
            for (int i = 0; i < cfg.k; ++i) p5 *= 5;
            if (cfg.k > 8 || cfg.kmer_lut_len != p5) return DNATOK_EINVAL;
            max_id = std::max<int64_t>(cfg.unk_id, cfg.pad_id);
            for (int64_t i = 0; i < p5; ++i) {
                if (cfg.kmer_lut[i] < 0) return DNATOK_EINVAL;
                max_id = std::max<int64_t>(max_id, cfg.kmer_lut[i]);
            }
            for (int i = 0; i < 5; ++i) max_id = std::max<int64_t>(max_id, cfg.nt_ids[i]);
        }
    } else {
        if (cfg.n_merges < 0 || cfg.n_merges > 65000 || (cfg.n_merges > 0 && !cfg.merges)) return DNATOK_EINVAL;
        max_id = std::max<int64_t>(max_id, std::max<int64_t>(cfg.n_id, cfg.base_id + 3 + cfg.n_merges));
    }
    if (cfg.id_dtype == DNATOK_I16 && max_id > 0x7fff) return DNATOK_EINVAL;

    // BPE rule table (validated before any device work; Q12)
    std::vector<uint64_t> table;
    uint32_t mask = 0;
    if (cfg.mode == DNATOK_BPE) {
        uint32_t size = 16;
        while (size < 2u * (uint32_t)cfg.n_merges + 1u) size <<= 1;
        mask = size - 1;
        table.assign(size, ~0ull);
        for (int32_t r = 0; r < cfg.n_merges; ++r) {
            int32_t L = cfg.merges[2 * r], R = cfg.merges[2 * r + 1];
            if (L < 0 || R < 0 || L >= 4 + r || R >= 4 + r) return DNATOK_EINVAL;
            uint32_t key = ((uint32_t)L << 16) | (uint32_t)R, hsh = host_hash(key) & mask;
            while (table[hsh] != ~0ull) {
                if ((uint32_t)(table[hsh] >> 32) == key) return DNATOK_EINVAL;   // duplicate pair
                hsh = (hsh + 1) & mask;
            }
            table[hsh] = ((uint64_t)key << 32) | (uint32_t)r;
        }
    }

    dnatok_t *h = new (std::nothrow) dnatok();
    if (!h) return DNATOK_ENOMEM;
    h->cfg = cfg; h->cfg.merges = nullptr; h->cfg.kmer_lut = nullptr; h->device = device;
    auto bail = [&](int code) { dnatok_destroy(h); return code; };
    DeviceGuard dev_guard_(device);
    if (!dev_guard_.ok) return bail(DNATOK_ECUDA);
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, device) != cudaSuccess) return bail(DNATOK_ECUDA);
    h->sm_count = prop.multiProcessorCount;
    h->d_static_rec_len = static_scratch_on(device);          // (the handle's device is current here)
    if (!h->d_static_rec_len) return bail(DNATOK_ECUDA);

    EncParams &p = h->prm;
    p.mode = cfg.mode == DNATOK_KMER ? MODE_KMER : MODE_SINGLE_NT;
    p.k = cfg.mode == DNATOK_KMER ? cfg.k : 1;
    p.tail_policy = cfg.tail_policy; p.strip_headers = cfg.strip_headers;
    p.unk_id = cfg.unk_id; p.base_id = cfg.base_id;
    for (int i = 0; i < 5; ++i) p.nt_ids[i] = cfg.nt_ids[i];
    p.four_k = cfg.mode == DNATOK_KMER ? (int32_t)(1ll << (2 * cfg.k)) : 0;
    p.fast_lut = 1;
    for (int i = 0; i < 4; ++i)
        if (cfg.class_lut[(uint8_t)"ACGT"[i]] != i || cfg.class_lut[(uint8_t)"acgt"[i]] != i) p.fast_lut = 0;
    p.fast_n = cfg.class_lut['N'] == DNATOK_CLS_N && cfg.class_lut['n'] == DNATOK_CLS_N;
    p.kmagic = p.k >= 2 ? (uint32_t)((1ull << 32) / (uint32_t)p.k) + 1u : 0u;
    p.kmer_lut = nullptr; p.remap4 = nullptr;
    if (cfg.kmer_lut) {
        // the id of every window of A, C, G, T comes from a 4^k-entry table derived here: remap4[code4] = kmer_lut[code5(code4)]
        const int k = cfg.k;
        const int64_t n4 = 1ll << (2 * k);
        std::vector<int32_t> remap((size_t)n4);
        for (int64_t c4 = 0; c4 < n4; ++c4) {
            int64_t c5 = 0;
            for (int i = k - 1; i >= 0; --i) c5 = c5 * 5 + ((c4 >> (2 * i)) & 3);
            remap[(size_t)c4] = cfg.kmer_lut[c5];
        }
        if (cudaMalloc(&h->d_kmer_lut, (size_t)cfg.kmer_lut_len * sizeof(int32_t)) != cudaSuccess ||
            cudaMalloc(&h->d_remap4, (size_t)n4 * sizeof(int32_t)) != cudaSuccess) return bail(DNATOK_ENOMEM);
        if (cudaMemcpy(h->d_kmer_lut, cfg.kmer_lut, (size_t)cfg.kmer_lut_len * sizeof(int32_t), cudaMemcpyHostToDevice) != cudaSuccess ||
            cudaMemcpy(h->d_remap4, remap.data(), (size_t)n4 * sizeof(int32_t), cudaMemcpyHostToDevice) != cudaSuccess)
            return bail(DNATOK_ECUDA);
        p.kmer_lut = h->d_kmer_lut; p.remap4 = h->d_remap4;
    }

    if (cudaMalloc(&h->d_lut, 256) != cudaSuccess) return bail(DNATOK_ENOMEM);
    if (cudaMemcpy(h->d_lut, cfg.class_lut, 256, cudaMemcpyHostToDevice) != cudaSuccess) return bail(DNATOK_ECUDA);
    if (cfg.mode == DNATOK_BPE) {
        h->table_mask = mask;
        if (cudaMalloc(&h->d_table, table.size() * sizeof(uint64_t)) != cudaSuccess) return bail(DNATOK_ENOMEM);
        if (cudaMemcpy(h->d_table, table.data(), table.size() * sizeof(uint64_t), cudaMemcpyHostToDevice) != cudaSuccess)
            return bail(DNATOK_ECUDA);
        // decode: spelling of every token (a base spells itself, token 4 + r = spelling(left) spelling(right)); kept on the
        // device unless the spellings add up to more than 64 MiB (then dnatok_decode is unavailable on this handle)
        {
            const int64_t V = 4 + (int64_t)cfg.n_merges;
            std::vector<uint32_t> off(V + 1, 0);
            std::vector<int64_t> len(V, 1);
            int64_t total = 4;
            bool fits = true;
            for (int32_t r = 0; r < cfg.n_merges && fits; ++r) {
                len[4 + r] = len[cfg.merges[2 * r]] + len[cfg.merges[2 * r + 1]];
                total += len[4 + r];
                fits = total <= (64ll << 20);
            }
            if (fits) {
                std::vector<uint8_t> pool((size_t)total);
                int64_t pos = 0;
                for (int64_t t = 0; t < V; ++t) {
                    off[t] = (uint32_t)pos;
                    if (t < 4) pool[pos] = (uint8_t)"ACGT"[t];
                    else {
                        const int32_t L = cfg.merges[2 * (t - 4)], R = cfg.merges[2 * (t - 4) + 1];
                        memcpy(&pool[pos], &pool[off[L]], (size_t)len[L]);
                        memcpy(&pool[pos + len[L]], &pool[off[R]], (size_t)len[R]);
                    }
                    pos += len[t];
                }
                off[V] = (uint32_t)pos;
                if (cudaMalloc(&h->d_spell_off, off.size() * sizeof(uint32_t)) != cudaSuccess ||
                    cudaMalloc(&h->d_spell, pool.size()) != cudaSuccess) return bail(DNATOK_ENOMEM);
                if (cudaMemcpy(h->d_spell_off, off.data(), off.size() * sizeof(uint32_t), cudaMemcpyHostToDevice) != cudaSuccess ||
                    cudaMemcpy(h->d_spell, pool.data(), pool.size(), cudaMemcpyHostToDevice) != cudaSuccess) return bail(DNATOK_ECUDA);
            }
        }
        // longest ACGT segment (run between N / UNK bytes) the merge kernels hold: up to 2048 symbols in the main kernel's
        // per-warp slice, up to BPE_GIANT_MAX in the giant kernel's (one warp per SM); longer ones are ECAPACITY
        int cap = (int)std::min<int64_t>(BPE_GIANT_MAX, std::max<int64_t>(BPE_SLOT_WORDS, (cfg.max_record_bytes + 63) & ~(int64_t)63));
        h->bpe_cap = cap;
        const int main_smem = BPE_WARPS * BPE_SLOT_WORDS * (int)sizeof(uint32_t);
        if (cudaFuncSetAttribute(bpe_merge_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, main_smem) != cudaSuccess)
            return bail(DNATOK_ECUDA);
        if (cap > BPE_SLOT_WORDS && cudaFuncSetAttribute(bpe_merge_giant_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                               cap * (int)sizeof(uint32_t)) != cudaSuccess) return bail(DNATOK_ECUDA);
        int nb = 0;
        cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, bpe_merge_kernel, BPE_WARPS * 32, main_smem);
        h->bpe_ctas_per_sm = std::max(nb, 1);
    }
    {
        // both encoders need more than the default 48 KiB of shared memory per CTA
#define DTK_V5(T) (const void *)v5::encode_tiles_v5<T, 0>, (const void *)v5::encode_tiles_v5<T, 1>, (const void *)v5::encode_tiles_v5<T, 2>, \
                  (const void *)v5::encode_tiles_v5<T, 3>, (const void *)v5::encode_tiles_v5<T, 4>, (const void *)v5::encode_tiles_v5<T, 5>, \
                  (const void *)v5::encode_tiles_v5<T, 6>, (const void *)v5::encode_tiles_v5<T, 8>, (const void *)v5::encode_tiles_v5<T, -1>
#define DTK_V7(T) (const void *)v7::encode_tiles_v7<T, 0, true>, (const void *)v7::encode_tiles_v7<T, 1, true>, (const void *)v7::encode_tiles_v7<T, 2, true>, \
                  (const void *)v7::encode_tiles_v7<T, 3, true>, (const void *)v7::encode_tiles_v7<T, 4, true>, (const void *)v7::encode_tiles_v7<T, 5, true>, \
                  (const void *)v7::encode_tiles_v7<T, 6, true>, (const void *)v7::encode_tiles_v7<T, 8, true>, (const void *)v7::encode_tiles_v7<T, -1, true>
        const void *k5[] = {DTK_V5(int32_t), DTK_V5(int16_t), (const void *)v5::encode_tiles_v5<uint8_t, 0>};
        const void *k7[] = {DTK_V7(int32_t), DTK_V7(int16_t), (const void *)v7::encode_tiles_v7<uint8_t, 0, true>};
#undef DTK_V5
#undef DTK_V7
        for (const void *kf : k5)
            if (cudaFuncSetAttribute(kf, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(v5::Smem5)) != cudaSuccess)
                return bail(DNATOK_ECUDA);
        for (const void *kf : k7)
            if (cudaFuncSetAttribute(kf, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(v7::Smem7)) != cudaSuccess)
                return bail(DNATOK_ECUDA);
#define DTK_FA(T) (const void *)fa::encode_fasta_kernel<T, 0>, (const void *)fa::encode_fasta_kernel<T, 1>, (const void *)fa::encode_fasta_kernel<T, 2>, \
                  (const void *)fa::encode_fasta_kernel<T, 3>, (const void *)fa::encode_fasta_kernel<T, 4>, (const void *)fa::encode_fasta_kernel<T, 5>, \
                  (const void *)fa::encode_fasta_kernel<T, 6>, (const void *)fa::encode_fasta_kernel<T, 8>, (const void *)fa::encode_fasta_kernel<T, -1>
#define DTK_FAF (const void *)fa::encode_fasta_kernel<int32_t, 0, true>, (const void *)fa::encode_fasta_kernel<int32_t, 1, true>, \
                (const void *)fa::encode_fasta_kernel<int32_t, 2, true>, (const void *)fa::encode_fasta_kernel<int32_t, 3, true>, \
                (const void *)fa::encode_fasta_kernel<int32_t, 4, true>, (const void *)fa::encode_fasta_kernel<int32_t, 5, true>, \
                (const void *)fa::encode_fasta_kernel<int32_t, 6, true>, (const void *)fa::encode_fasta_kernel<int32_t, 8, true>, \
                (const void *)fa::encode_fasta_kernel<int32_t, -1, true>
        const void *kfa[] = {DTK_FA(int32_t), DTK_FA(int16_t), DTK_FAF, (const void *)fa::encode_fasta_kernel<uint8_t, 0>};
#undef DTK_FA
        for (const void *kf : kfa)
            if (cudaFuncSetAttribute(kf, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(fa::SmemFa)) != cudaSuccess)
                return bail(DNATOK_ECUDA);
        int nb = 0;
        cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, fa::encode_fasta_kernel<int32_t, -1>, fa::FW_WARPS * 32, sizeof(fa::SmemFa));
        h->fasta_ctas_per_sm = std::max(nb, 1);
        cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, v5::encode_tiles_v5<int32_t, -1>, NT, sizeof(v5::Smem5));
        h->enc_ctas_per_sm = std::max(nb, 1);
        cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, v7::encode_tiles_v7<int32_t, -1, true>, v7::NT7, sizeof(v7::Smem7));
        h->dense_ctas_per_sm = std::max(nb, 1);
        h->dense = !cfg.strip_headers;
        for (int b = 0; b < 256; ++b) if (cfg.class_lut[b] == DNATOK_CLS_SKIP) h->dense = false;
    }
    if (ctx_init(h, h->ctx) != DNATOK_OK) return bail(DNATOK_ECUDA);
    *out = h;
    return DNATOK_OK;
}

int dnatok_destroy(dnatok_t *h) {
    if (!h) return DNATOK_OK;
    DeviceGuard dev_guard_(h->device);
    cudaDeviceSynchronize();
    ring_free(h->ring);
    ctx_free(h->ctx);
    cudaFree(h->d_lut); cudaFree(h->d_table); cudaFree(h->d_spell_off); cudaFree(h->d_spell); cudaFree(h->d_rec_len); cudaFree(h->d_kmer_lut); cudaFree(h->d_remap4);
    delete h;
    return DNATOK_OK;
}

int dnatok_encode(dnatok_t *h, const uint8_t *d_bytes, int64_t n_bytes, const int64_t *d_rec_offsets,
                  int64_t n_records, void *d_ids_out, int64_t ids_capacity, int64_t *d_out_offsets, void *stream) {
    if (!h) return DNATOK_EINVAL;
    if (n_bytes < 0 || n_records < 0 || ids_capacity < 0 || !d_rec_offsets || !d_out_offsets ||
        (n_bytes > 0 && !d_bytes) || (ids_capacity > 0 && !d_ids_out))
        return fail(h, DNATOK_EINVAL, "dnatok_encode: bad argument");
    USE_DEVICE(h);
    return encode_on(h, h->ctx, d_bytes, n_bytes, d_rec_offsets, n_records, 0, d_ids_out, ids_capacity,
                     d_out_offsets, (cudaStream_t)stream);
}

int dnatok_encode_pad(dnatok_t *h, const uint8_t *d_bytes, int64_t n_bytes, const int64_t *d_rec_offsets,
                      int64_t n_records, void *d_ids_out, int64_t ids_capacity, int64_t *d_out_offsets,
                      int32_t *d_batch_ids, uint8_t *d_mask, void *stream) {
    if (!h) return DNATOK_EINVAL;
    if (h->cfg.seq_len <= 0) return fail(h, DNATOK_EINVAL, "dnatok_encode_pad: handle was created with seq_len == 0");
    if (n_bytes < 0 || n_records < 0 || ids_capacity < 0 || !d_rec_offsets || !d_out_offsets ||
        (n_bytes > 0 && !d_bytes) || (ids_capacity > 0 && !d_ids_out) || (n_records > 0 && !d_batch_ids))
        return fail(h, DNATOK_EINVAL, "dnatok_encode_pad: bad argument");
    USE_DEVICE(h);
    bool fused = false;
    int rc = encode_on(h, h->ctx, d_bytes, n_bytes, d_rec_offsets, n_records, 0, d_ids_out, ids_capacity, d_out_offsets,
                       (cudaStream_t)stream, d_batch_ids, d_mask, &fused);
    if (rc || fused) return rc;
    return pad_on(h, d_ids_out, d_out_offsets, n_records, d_batch_ids, d_mask, (cudaStream_t)stream, ids_capacity);
}

int dnatok_pad(dnatok_t *h, const void *d_ids, const int64_t *d_out_offsets, int64_t n_records,
               int32_t *d_batch_ids, uint8_t *d_mask, void *stream) {
    if (!h) return DNATOK_EINVAL;
    if (h->cfg.seq_len <= 0) return fail(h, DNATOK_EINVAL, "dnatok_pad: handle was created with seq_len == 0");
    if (n_records < 0 || !d_out_offsets || (n_records > 0 && !d_batch_ids))
        return fail(h, DNATOK_EINVAL, "dnatok_pad: bad argument");
    USE_DEVICE(h);
    return pad_on(h, d_ids, d_out_offsets, n_records, d_batch_ids, d_mask, (cudaStream_t)stream);
}

// The chunk loop of step 7.  h_pinned != NULL: the ring's host slots alias the caller's page-locked buffer.  Otherwise every
// chunk is produced by fill(fill_user, chunk_index, offset, n_bytes, dst) into one of n_streams + 1 pinned staging slots
// (PAPER.md:181 persistent pinned buffers) and copied to the device from there.  Any failure returns at once; the caller
// drains the streams.
static int stream_run(dnatok_t *h, const uint8_t *h_pinned, dnatok_fill_fn fill, void *fill_user, int64_t n_bytes,
                      const int64_t *h_rec_offsets, int64_t n_records, dnatok_batch_fn on_batch, void *user) {
    StreamRing &R = h->ring;
    const int64_t C = R.chunk_bytes;
    const int64_t n_chunks = std::max<int64_t>(1, (n_bytes + C - 1) / C);
    const int n_stage = (int)R.stage.size();
    int rc;
    int64_t ra = 0;                                   // first record not yet delivered
    for (int64_t i = 0; i < n_chunks; ++i) {
        StreamSlot &S = R.slots[i % R.n_slots];
        cudaStream_t st = R.streams[i % R.n_streams];
        const int64_t c0 = i * C, c1 = std::min(n_bytes, c0 + C);
        // records that end in this chunk: h_rec_offsets[r + 1] in (c0, c1] (all the rest in the last chunk)
        int64_t rb;
        if (i == n_chunks - 1) rb = n_records;
        else rb = std::upper_bound(h_rec_offsets + ra + 1, h_rec_offsets + n_records + 1, c1) - h_rec_offsets - 1;
        if (rb < ra) rb = ra;
        const int64_t rows = rb - ra;
        if (rows > R.max_rows)
            return fail(h, DNATOK_ECAPACITY, "chunk %lld holds %lld records > max_rows_per_chunk %lld",
                        (long long)i, (long long)rows, (long long)R.max_rows);
        // bytes of the record cut by the previous boundary live in the previous slot's buffer
        const int64_t data0 = std::min(h_rec_offsets[ra], c0);       // host offset of the first byte needed
        const int64_t carry = c0 - data0;
        if (carry > R.carry_cap)
            return fail(h, DNATOK_ECAPACITY, "record %lld needs %lld carried bytes > max_record_bytes %lld",
                        (long long)ra, (long long)carry, (long long)R.carry_cap);
        // the producer fills its staging slot while earlier chunks are still in flight
        const uint8_t *src = h_pinned ? h_pinned + c0 : nullptr;
        if (!h_pinned && c1 > c0) {
            const int sl = (int)(i % n_stage);
            CU(cudaEventSynchronize(R.ev_stage[sl]));                 // the copy out of its previous use has finished
            if (fill(fill_user, i, c0, c1 - c0, R.stage[sl]) != 0)
                return fail(h, DNATOK_EINVAL, "dnatok_stream_encode_from: the producer failed on chunk %lld", (long long)i);
            src = R.stage[sl];
        }
        uint8_t *d_chunk = S.d_buf + R.carry_cap;
        // this buffer was last used by chunk i - n_slots (same stream only if n_slots == n_streams) and read by
        // chunk i - n_slots + 1's carry copy
        if (i >= R.n_slots) {
            CU(cudaStreamWaitEvent(st, S.ev_done, 0));
            CU(cudaStreamWaitEvent(st, R.slots[(i + 1) % R.n_slots].ev_carry, 0));
        }
        if (carry > 0) {
            StreamSlot &Pv = R.slots[(i - 1) % R.n_slots];
            CU(cudaStreamWaitEvent(st, Pv.ev_h2d, 0));
            CU(cudaMemcpyAsync(d_chunk - carry, Pv.d_buf + R.carry_cap + (data0 - (c0 - C)), (size_t)carry,
                               cudaMemcpyDeviceToDevice, st));
        }
        CU(cudaEventRecord(S.ev_carry, st));
        if (c1 > c0) CU(cudaMemcpyAsync(d_chunk, src, (size_t)(c1 - c0), cudaMemcpyHostToDevice, st));
        CU(cudaEventRecord(S.ev_h2d, st));
        if (!h_pinned && c1 > c0) CU(cudaEventRecord(R.ev_stage[i % n_stage], st));
        // record offsets of this batch (staged through the slot's pinned buffer)
        CU(cudaEventSynchronize(S.ev_off));
        memcpy(S.h_recoff, h_rec_offsets + ra, (size_t)(rows + 1) * sizeof(int64_t));
        CU(cudaMemcpyAsync(S.d_recoff, S.h_recoff, (size_t)(rows + 1) * sizeof(int64_t), cudaMemcpyHostToDevice, st));
        CU(cudaEventRecord(S.ev_off, st));
        // encode the whole records [ra, rb): buffer starts at host offset data0
        const int64_t nb = std::max<int64_t>(0, (rows > 0 ? h_rec_offsets[rb] : data0) - data0);
        // (encode, then pad: a batch hands out its CSR ids as well as its rows, so the fused call of dnatok_encode_pad, which
        // leaves the ids unwritten, is not used here -- and a chunk's kernels are a tenth of its host-to-device copy anyway)
        rc = encode_on(h, S.ctx, d_chunk - carry, nb, S.d_recoff, rows, data0, S.d_ids, R.carry_cap + C,
                       S.d_out_off, st);
        if (rc) return rc;
        if (h->cfg.seq_len > 0) {
            rc = pad_on(h, S.d_ids, S.d_out_off, rows, S.d_batch, S.d_mask, st, R.carry_cap + C);
            if (rc) return rc;
        }
        if (on_batch) {
            dnatok_batch b;
            b.first_record = ra; b.n_records = rows; b.d_ids = S.d_ids; b.d_out_offsets = S.d_out_off;
            b.d_batch_ids = h->cfg.seq_len > 0 ? S.d_batch : nullptr;
            b.d_mask = h->cfg.seq_len > 0 ? S.d_mask : nullptr;
            b.chunk_index = i; b.stream = (void *)st;
            on_batch(user, &b);
        }
        CU(cudaEventRecord(S.ev_done, st));
        ra = rb;
    }
    for (auto st : R.streams) CU(cudaStreamSynchronize(st));
    for (auto &sl : R.slots) { rc = status_of(h, sl.ctx); if (rc) return rc; }
    return DNATOK_OK;
}

static int stream_entry(dnatok_t *h, const uint8_t *h_pinned, dnatok_fill_fn fill, void *fill_user, int64_t n_bytes,
                        const int64_t *h_rec_offsets, int64_t n_records, int64_t chunk_bytes, int n_streams,
                        int64_t max_rows_per_chunk, dnatok_batch_fn on_batch, void *user) {
    if (max_rows_per_chunk <= 0) max_rows_per_chunk = chunk_bytes / 64 + 2;
    int rc = ring_setup(h, chunk_bytes, n_streams, max_rows_per_chunk);
    if (rc == DNATOK_OK && !h_pinned) rc = ring_stage_setup(h);
    if (rc == DNATOK_OK) rc = stream_run(h, h_pinned, fill, fill_user, n_bytes, h_rec_offsets, n_records, on_batch, user);
    if (rc != DNATOK_OK) {
        // nothing stays in flight behind a failed call: the ring's streams are drained and a sticky CUDA error is cleared
        for (auto st : h->ring.streams) cudaStreamSynchronize(st);
        cudaGetLastError();
    }
    return rc;
}

static int fill_from_memory(void *user, int64_t, int64_t offset, int64_t n, uint8_t *dst) {
    memcpy(dst, static_cast<const uint8_t *>(user) + offset, (size_t)n);
    return 0;
}

int dnatok_stream_encode(dnatok_t *h, const uint8_t *h_bytes, int64_t n_bytes, const int64_t *h_rec_offsets,
                         int64_t n_records, int64_t chunk_bytes, int n_streams, int64_t max_rows_per_chunk,
                         dnatok_batch_fn on_batch, void *user) {
    if (!h) return DNATOK_EINVAL;
    if (n_bytes < 0 || n_records < 0 || !h_rec_offsets || chunk_bytes <= 0 || n_streams < 1 || n_streams > 64 ||
        (n_bytes > 0 && !h_bytes))
        return fail(h, DNATOK_EINVAL, "dnatok_stream_encode: bad argument");
    USE_DEVICE(h);
    bool pinned = n_bytes == 0;
    if (n_bytes > 0) {
        cudaPointerAttributes at;
        cudaError_t e = cudaPointerGetAttributes(&at, h_bytes);
        if (e != cudaSuccess) cudaGetLastError();
        else if (at.type == cudaMemoryTypeDevice || at.type == cudaMemoryTypeManaged)
            return fail(h, DNATOK_EINVAL, "dnatok_stream_encode: h_bytes is not host memory");
        pinned = e == cudaSuccess && at.type == cudaMemoryTypeHost;
    }
    // page-locked input: the ring's host slots alias it; pageable input goes through the pinned staging ring
    return stream_entry(h, pinned ? h_bytes : nullptr, fill_from_memory, const_cast<uint8_t *>(h_bytes), n_bytes, h_rec_offsets,
                        n_records, chunk_bytes, n_streams, max_rows_per_chunk, on_batch, user);
}

int dnatok_stream_encode_from(dnatok_t *h, dnatok_fill_fn fill, void *fill_user, int64_t n_bytes,
                              const int64_t *h_rec_offsets, int64_t n_records, int64_t chunk_bytes, int n_streams,
                              int64_t max_rows_per_chunk, dnatok_batch_fn on_batch, void *user) {
    if (!h) return DNATOK_EINVAL;
    if (!fill || n_bytes < 0 || n_records < 0 || !h_rec_offsets || chunk_bytes <= 0 || n_streams < 1 || n_streams > 64)
        return fail(h, DNATOK_EINVAL, "dnatok_stream_encode_from: bad argument");
    USE_DEVICE(h);
    return stream_entry(h, nullptr, fill, fill_user, n_bytes, h_rec_offsets, n_records, chunk_bytes, n_streams,
                        max_rows_per_chunk, on_batch, user);
}

int dnatok_check(dnatok_t *h, void *stream) {
    if (!h) return DNATOK_EINVAL;
    USE_DEVICE(h);
    CU(cudaStreamSynchronize((cudaStream_t)stream));
    return status_of(h, h->ctx);
}

int dnatok_set_super_tile(dnatok_t *h, int32_t sub_tiles) {
    if (!h) return DNATOK_EINVAL;
    if (sub_tiles < 0 || sub_tiles > S_MAX) return fail(h, DNATOK_EINVAL, "dnatok_set_super_tile: sub_tiles must be in 0..%d", S_MAX);
    h->force_S = sub_tiles;
    return DNATOK_OK;
}

int dnatok_set_fast_path(dnatok_t *h, int32_t enable) {
    if (!h) return DNATOK_EINVAL;
    if (enable < 0 || enable > 2) return fail(h, DNATOK_EINVAL, "dnatok_set_fast_path: 0, 1 or 2");
    h->fast_path = enable;
    return DNATOK_OK;
}

int dnatok_fast_path_taken(dnatok_t *h, void *stream) {
    if (!h) return DNATOK_EINVAL;
    USE_DEVICE(h);
    CU(cudaStreamSynchronize((cudaStream_t)stream));
    if (!h->ctx.fa_tried) return 0;
    uint32_t flag = 0;
    CU(cudaMemcpy(&flag, h->ctx.fa_flag, sizeof(flag), cudaMemcpyDeviceToHost));
    return flag == 0u ? 1 : 0;
}

int dnatok_set_grid_cap(dnatok_t *h, int32_t max_ctas) {
    if (!h) return DNATOK_EINVAL;
    if (max_ctas < 0) return fail(h, DNATOK_EINVAL, "dnatok_set_grid_cap: max_ctas must be >= 0");
    h->grid_cap = max_ctas;
    return DNATOK_OK;
}

#ifdef DTK_PROF
// debug builds only: read and clear the phase timers of the handle's resident-encode context
int dnatok_debug_prof(dnatok_t *h, unsigned long long *out64) {
    cudaDeviceSynchronize();
    cudaMemcpy(out64, h->ctx.prof, 64 * sizeof(unsigned long long), cudaMemcpyDeviceToHost);
    cudaMemset(h->ctx.prof, 0, 64 * sizeof(unsigned long long));
    return DNATOK_OK;
}
#endif

const char *dnatok_last_error(const dnatok_t *h) { return h ? h->err.c_str() : "null handle"; }

// ---- reverse complement, decode, embedding gather, widening ------------------------------------
int dnatok_revcomp(dnatok_t *h, const uint8_t *d_bytes, int64_t n_bytes, const int64_t *d_rec_offsets, int64_t n_records,
                   uint8_t *d_out, void *stream) {
    if (!h) return DNATOK_EINVAL;
    if (n_bytes < 0 || n_records < 0 || !d_rec_offsets || (n_bytes > 0 && (!d_bytes || !d_out)) || d_bytes == d_out)
        return fail(h, DNATOK_EINVAL, "dnatok_revcomp: bad argument (in-place is not supported)");
    if (n_bytes == 0) return DNATOK_OK;
    USE_DEVICE(h);
    RevcompArgs a{d_bytes, d_out, d_rec_offsets, n_records, n_bytes};
    const int64_t n16 = (n_bytes + 15) >> 4;
    int grid = (int)std::min<int64_t>((n16 + 255) / 256, (int64_t)h->sm_count * 8);
    if (h->grid_cap > 0) grid = std::min(grid, h->grid_cap);
    revcomp_kernel<<<grid, 256, 0, (cudaStream_t)stream>>>(a);
    CU(cudaGetLastError());
    h->launches += 1;
    return DNATOK_OK;
}

int dnatok_decode(dnatok_t *h, const void *d_ids, const int64_t *d_out_offsets, int64_t n_records, uint8_t *d_bytes_out,
                  int64_t bytes_capacity, int64_t *d_byte_offsets, void *stream) {
    if (!h) return DNATOK_EINVAL;
    if (n_records < 0 || bytes_capacity < 0 || !d_out_offsets || !d_byte_offsets || (bytes_capacity > 0 && !d_bytes_out))
        return fail(h, DNATOK_EINVAL, "dnatok_decode: bad argument");
    if (h->d_remap4) return fail(h, DNATOK_EINVAL, "dnatok_decode: a handle with a k-mer id table has no inverse table");
    if (h->cfg.mode == DNATOK_BPE && !h->d_spell)
        return fail(h, DNATOK_EINVAL, "dnatok_decode: the merge table's token spellings exceed 64 MiB");
    USE_DEVICE(h);
    cudaStream_t st = (cudaStream_t)stream;
    if (n_records + 1 > h->rec_len_cap) {
        if (h->d_rec_len) CU(cudaFreeAsync(h->d_rec_len, st));
        h->d_rec_len = nullptr; h->rec_len_cap = 0;
        const int64_t cap = n_records + n_records / 4 + 256;
        CU(cudaMallocAsync((void **)&h->d_rec_len, (size_t)cap * sizeof(int32_t), st));
        h->rec_len_cap = cap;
    }
    const dnatok_config &cfg = h->cfg;
    DecodeArgs a;
    a.ids = d_ids; a.out_off = d_out_offsets; a.n_rec = n_records;
    a.mode = cfg.mode; a.k = cfg.mode == DNATOK_KMER ? cfg.k : 1; a.base_id = cfg.base_id; a.n_id = cfg.n_id; a.pad_id = cfg.pad_id;
    for (int i = 0; i < 5; ++i) a.nt_ids[i] = cfg.nt_ids[i];
    a.four_k = 1ll << (2 * a.k);
    a.n_tokens_bpe = 4 + cfg.n_merges; a.spell_off = h->d_spell_off; a.spell = h->d_spell;
    a.rec_len = h->d_rec_len; a.byte_off = d_byte_offsets; a.out = d_bytes_out; a.out_cap = bytes_capacity;
    a.status = h->ctx.d_status;
    int grid = (int)std::min<int64_t>((n_records + 7) / 8 + 1, (int64_t)h->sm_count * 8);
    if (h->grid_cap > 0) grid = std::min(grid, h->grid_cap);
    const bool i16 = cfg.id_dtype == DNATOK_I16;
    if (i16) decode_kernel<int16_t, false><<<grid, 256, 0, st>>>(a); else decode_kernel<int32_t, false><<<grid, 256, 0, st>>>(a);
    scan_counts_kernel<<<1, 1024, 0, st>>>(h->d_rec_len, n_records, d_byte_offsets);
    if (i16) decode_kernel<int16_t, true><<<grid, 256, 0, st>>>(a); else decode_kernel<int32_t, true><<<grid, 256, 0, st>>>(a);
    CU(cudaGetLastError());
    h->launches += 3;
    return DNATOK_OK;
}

// dnatok_decode without any allocation: the per-record lengths live in the library's static device array.  Nothing in it has
// to start at zero (the length pass writes every entry the scan reads), so stale contents of an earlier call do no harm; two
// calls that overlap on the GPU would race on it.
int dnatok_decode_static(dnatok_t *h, const void *d_ids, const int64_t *d_out_offsets, int64_t n_records, uint8_t *d_bytes_out,
                         int64_t bytes_capacity, int64_t *d_byte_offsets, void *stream) {
    if (!h) return DNATOK_EINVAL;
    if (n_records < 0 || bytes_capacity < 0 || !d_out_offsets || !d_byte_offsets || (bytes_capacity > 0 && !d_bytes_out))
        return fail(h, DNATOK_EINVAL, "dnatok_decode_static: bad argument");
    if (n_records > DNATOK_DECODE_STATIC_MAX_RECORDS)
        return fail(h, DNATOK_ECAPACITY, "dnatok_decode_static: %lld records exceed the static scratch's %d (use dnatok_decode, or split the call)",
                    (long long)n_records, (int)DNATOK_DECODE_STATIC_MAX_RECORDS);
    if (h->d_remap4) return fail(h, DNATOK_EINVAL, "dnatok_decode_static: a handle with a k-mer id table has no inverse table");
    if (h->cfg.mode == DNATOK_BPE && !h->d_spell)
        return fail(h, DNATOK_EINVAL, "dnatok_decode_static: the merge table's token spellings exceed 64 MiB");
    USE_DEVICE(h);
    cudaStream_t st = (cudaStream_t)stream;
    const dnatok_config &cfg = h->cfg;
    DecodeArgs a;
    a.ids = d_ids; a.out_off = d_out_offsets; a.n_rec = n_records;
    a.mode = cfg.mode; a.k = cfg.mode == DNATOK_KMER ? cfg.k : 1; a.base_id = cfg.base_id; a.n_id = cfg.n_id; a.pad_id = cfg.pad_id;
    for (int i = 0; i < 5; ++i) a.nt_ids[i] = cfg.nt_ids[i];
    a.four_k = 1ll << (2 * a.k);
    a.n_tokens_bpe = 4 + cfg.n_merges; a.spell_off = h->d_spell_off; a.spell = h->d_spell;
    a.rec_len = h->d_static_rec_len; a.byte_off = d_byte_offsets; a.out = d_bytes_out; a.out_cap = bytes_capacity;
    a.status = h->ctx.d_status;
    int grid = (int)std::min<int64_t>((n_records + 7) / 8 + 1, (int64_t)h->sm_count * 8);
    if (h->grid_cap > 0) grid = std::min(grid, h->grid_cap);
    const bool i16 = cfg.id_dtype == DNATOK_I16;
    if (i16) decode_kernel<int16_t, false><<<grid, 256, 0, st>>>(a); else decode_kernel<int32_t, false><<<grid, 256, 0, st>>>(a);
    scan_counts_kernel<<<1, 1024, 0, st>>>(h->d_static_rec_len, n_records, d_byte_offsets);
    if (i16) decode_kernel<int16_t, true><<<grid, 256, 0, st>>>(a); else decode_kernel<int32_t, true><<<grid, 256, 0, st>>>(a);
    CU(cudaGetLastError());
    h->launches += 3;
    return DNATOK_OK;
}

int64_t dnatok_microbatch_rows(int64_t b_emb, int64_t m_tokens, int64_t t_len) {
    int64_t q = t_len > 0 ? m_tokens / t_len : m_tokens;
    if (q < 1) q = 1;
    return b_emb < q ? b_emb : q;
}

int dnatok_embed(dnatok_t *h, const int32_t *d_ids, int64_t n_rows, int64_t t_len, const void *d_table, int64_t vocab,
                 int64_t row_bytes, void *d_out, int64_t b_emb, int64_t m_tokens, dnatok_microbatch_fn on_microbatch,
                 void *user, void *stream) {
    if (!h) return DNATOK_EINVAL;
    if (n_rows < 0 || t_len <= 0 || vocab <= 0 || row_bytes <= 0 || (row_bytes & 3) || b_emb <= 0 || m_tokens <= 0 ||
        row_bytes > (1 << 20) || (n_rows > 0 && (!d_ids || !d_table || !d_out)) ||
        (reinterpret_cast<uintptr_t>(d_table) & 3) || (reinterpret_cast<uintptr_t>(d_out) & 3))
        return fail(h, DNATOK_EINVAL, "dnatok_embed: bad argument (row_bytes must be a multiple of 4, buffers 4-byte aligned)");
    USE_DEVICE(h);
    const bool v16 = (row_bytes & 15) == 0 && (reinterpret_cast<uintptr_t>(d_table) & 15) == 0 &&
                     (reinterpret_cast<uintptr_t>(d_out) & 15) == 0;
    const int64_t b = dnatok_microbatch_rows(b_emb, m_tokens, t_len);
    for (int64_t r0 = 0; r0 < n_rows; r0 += b) {
        const int64_t rows = std::min(b, n_rows - r0), toks = rows * t_len;
        const int64_t acc = toks * (row_bytes / (v16 ? 16 : 4));
        int grid = (int)std::min<int64_t>((acc + 255) / 256, (int64_t)h->sm_count * 16);
        if (h->grid_cap > 0) grid = std::min(grid, h->grid_cap);
        uint8_t *out = reinterpret_cast<uint8_t *>(d_out) + r0 * t_len * row_bytes;
        if (v16) embed_kernel<16><<<grid, 256, 0, (cudaStream_t)stream>>>(d_ids + r0 * t_len, toks, (const uint8_t *)d_table, vocab, (int32_t)row_bytes, out);
        else embed_kernel<4><<<grid, 256, 0, (cudaStream_t)stream>>>(d_ids + r0 * t_len, toks, (const uint8_t *)d_table, vocab, (int32_t)row_bytes, out);
        CU(cudaGetLastError());
        h->launches += 1;
        if (on_microbatch) on_microbatch(user, r0, rows, out, stream);
    }
    return DNATOK_OK;
}

int dnatok_widen_ids(dnatok_t *h, const int32_t *d_ids, int64_t n, int64_t *d_out, void *stream) {
    if (!h) return DNATOK_EINVAL;
    if (n < 0 || (n > 0 && (!d_ids || !d_out))) return fail(h, DNATOK_EINVAL, "dnatok_widen_ids: bad argument");
    if (n == 0) return DNATOK_OK;
    USE_DEVICE(h);
    int grid = (int)std::min<int64_t>((n / 4 + 255) / 256 + 1, (int64_t)h->sm_count * 8);
    if (h->grid_cap > 0) grid = std::min(grid, h->grid_cap);
    widen_kernel<<<grid, 256, 0, (cudaStream_t)stream>>>(d_ids, n, d_out);
    CU(cudaGetLastError());
    h->launches += 1;
    return DNATOK_OK;
}

int64_t dnatok_launch_count(const dnatok_t *h) { return h ? h->launches : 0; }

}  // extern "C"
