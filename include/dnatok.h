/*
 * dnatok.h -- C-ABI of the B200-native DNATok hot path.
 *
 * Raw ASCII DNA bytes (FASTA-style records) -> token-ID streams on one GPU:
 * 256-entry byte LUT (section 2.2 "bytes path"; Algorithm 1),
 * newline / header stripping, then one of three vocabulary-agnostic encoders
 * (single-nucleotide; non-overlapping k-mer, "length k, stride k", Alg. 1
 * l.18 and PAPER.md:115-117 Alg. 2 l.7-8; BPE), CSR offsets,
 * optional padding + attention mask (Alg. 2 l.12-14), and a pinned,
 * multi-stream scheduler that overlaps the H2D copy of chunk i+1 with the encode of
 * chunk i (section 2.2 "Pipelined streaming").  Everything the
 * paper leaves open follows BASELINE.json north_star and the readings Q1-Q26 of
 * SURVEY.md section 8(c), restated in DESIGN.md.
 *
 * Conventions
 *   - plain C, no CUDA or torch types: a stream is passed as `void *` holding a
 *     cudaStream_t (NULL = the legacy default stream); pointers named d_* are DEVICE
 *     pointers, h_* are HOST pointers.
 *   - every function returns a dnatok_status; nothing is thrown across the ABI.
 *     dnatok_last_error() gives a human-readable message for the last failure on a
 *     handle.
 *   - the caller owns every input and output buffer.  The handle owns only what it
 *     allocates itself (LUT copy, merge-rule hash, scan scratch, streaming slots);
 *     dnatok_destroy() frees all of it.
 *   - calls on ONE handle must be ordered with respect to each other (same stream, or
 *     explicit event dependencies): the handle's scan scratch is not re-entrant.  Use
 *     one handle per concurrent stream.
 *   - there is no CPU fallback: every step runs in CUDA kernels for sm_100a.
 *
 * Class codes used by class_lut: 0..3 = A,C,G,T; 4 = N; 5 = UNK; 255 = SKIP (dropped).
 */
#ifndef DNATOK_H
#define DNATOK_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct dnatok dnatok_t;   /* opaque */

typedef enum {
    DNATOK_OK = 0,
    DNATOK_EINVAL = 1,      /* bad argument or configuration                                    */
    DNATOK_ENOMEM = 2,      /* host or device allocation failed                                 */
    DNATOK_ECUDA = 3,       /* a CUDA runtime call failed; see dnatok_last_error()              */
    DNATOK_ECAPACITY = 4,   /* an output or carry buffer was too small; nothing written past it */
    DNATOK_ESTATE = 5       /* internal scan protocol failure (look-back spin limit hit)        */
} dnatok_status;

enum { DNATOK_SINGLE_NT = 0, DNATOK_KMER = 1, DNATOK_BPE = 2 };               /* mode        */
enum { DNATOK_I16 = 2, DNATOK_I32 = 4 };                                      /* id_dtype    */
enum { DNATOK_TAIL_PER_BASE = 0, DNATOK_TAIL_DROP = 1, DNATOK_TAIL_UNK = 2 }; /* tail_policy */
enum { DNATOK_PAD_LEFT = 0, DNATOK_PAD_RIGHT = 1 };                           /* pad_side    */

#define DNATOK_CLS_N    4
#define DNATOK_CLS_UNK  5
#define DNATOK_CLS_SKIP 255
#define DNATOK_MAX_K    15

/*
 * Create-time specification (vocabulary / LUT spec, k or merge table).
 * Zero-initialise, set struct_size = sizeof(dnatok_config), then call
 * dnatok_config_default() or fill the fields by hand.
 */
typedef struct {
    uint32_t struct_size;     /* sizeof(dnatok_config); versioning                                         */
    int32_t  mode;            /* DNATOK_SINGLE_NT | DNATOK_KMER | DNATOK_BPE                                */
    int32_t  k;               /* KMER: window length 1..15 (ignored otherwise)                             */
    int32_t  id_dtype;        /* DNATOK_I16 | DNATOK_I32: element type of ids_out.  I16 needs max id < 2^15 */
    uint8_t  class_lut[256];  /* byte -> class code; all-zero => the default table (Aa Cc Gg Tt -> 0..3,    */
                              /* Nn -> 4, '\n' '\r' -> SKIP, every other byte -> UNK)                       */
    int32_t  strip_headers;   /* != 0: a line whose first byte is '>' is dropped through its '\n' (Q4).     */
                              /* Requires class_lut['\n'] == SKIP.                                          */
    int32_t  pad_id;          /* 0                                                                          */
    int32_t  unk_id;          /* 1                                                                          */
    int32_t  nt_ids[5];       /* SINGLE_NT: ids of A,C,G,T,N (2,3,4,5,6)                                    */
    int32_t  base_id;         /* KMER: id = base_id + packed code; BPE: id = base_id + token (3)            */
    int32_t  n_id;            /* BPE: id of an N byte (2)                                                   */
    int32_t  tail_policy;     /* KMER: what the n mod k trailing bases become (Q9)                          */
    const int32_t *merges;    /* BPE: HOST pointer to n_merges (left,right) pairs, copied at create;        */
    int32_t  n_merges;        /*      rule r produces token 4 + r; parts must be < 4 + r, pairs unique (Q12) */
    int32_t  seq_len;         /* pad: row length of batch_ids / mask; 0 => dnatok_pad unavailable           */
    int32_t  pad_side;        /* DNATOK_PAD_LEFT (paper) | DNATOK_PAD_RIGHT                   */
    int64_t  max_record_bytes;/* streaming: longest record in bytes the carry buffer must hold; BPE: longest */
                              /* ACGT run between two N / UNK bytes the merge workspace must hold (runs of   */
                              /* up to 2048 symbols always fit, at most 49152); 0 => 1 MiB                   */
    const int32_t *kmer_lut;  /* KMER, optional (NULL: ids are the base-4 closed form): HOST pointer to the    */
    int64_t  kmer_lut_len;    /* paper's kmer_lut[0..5^k-1] (Alg. 1 l.18-22), copied at create;   */
                              /* must be 5^k, k <= 8.  A window's id is kmer_lut[sum_i digit_i * 5^(k-1-i)],  */
                              /* digit = 0..3 for A,C,G,T and 4 for N and any other kept byte, so the table   */
                              /* decides what a window holding N becomes; PER_BASE tail bases get nt_ids[c].  */
} dnatok_config;

/* Fill *cfg with the BASELINE.json vocabulary (PAD 0, UNK 1, A..T 2..5, N 6; k-mer/BPE base_id 3, n_id 2),
 * default LUT, strip_headers = 1, I32, PER_BASE tail, LEFT pad, seq_len 0.  mode and k as given.          */
void dnatok_config_default(dnatok_config *cfg, int32_t mode, int32_t k);

/*
 * dnatok_create: validate cfg, select `device`, upload LUT / merge table, allocate scan scratch.
 * EINVAL: k outside 1..15 (KMER); max id not fitting id_dtype; BPE rule referring to a token >= its own
 * product or a duplicate pair; seq_len < 0; strip_headers with class_lut['\n'] != SKIP; class_lut entry
 * not in {0..5, 255}; kmer_lut given with mode != KMER, k > 8, kmer_lut_len != 5^k or an id not fitting id_dtype.
 * On success *out owns the handle.
 */
int dnatok_create(const dnatok_config *cfg, int device, dnatok_t **out);
int dnatok_destroy(dnatok_t *h);

/*
 * dnatok_encode: steps 1-5 (classify, strip, encode, CSR offsets) for n_records records.
 *   d_bytes        [n_bytes] uint8, any alignment.  Record r is the byte range
 *                  [d_rec_offsets[r], d_rec_offsets[r+1]).
 *   d_rec_offsets  [n_records+1] int64, non-decreasing, 0 <= offsets[0], offsets[n_records] <= n_bytes
 *                  (precondition, not checked).  Bytes outside every record are ignored.
 *   d_ids_out      [ids_capacity] elements of id_dtype.  ids_capacity >= n_bytes always suffices
 *                  (tokens <= kept bases <= bytes).  On overflow nothing is written past the end, the
 *                  handle's status word is set and dnatok_check() returns DNATOK_ECAPACITY.
 *   d_out_offsets  [n_records+1] int64: exclusive prefix sum of per-record token counts, total last.
 * Only enqueues work on `stream`; never synchronises.
 */
int dnatok_encode(dnatok_t *h, const uint8_t *d_bytes, int64_t n_bytes,
                  const int64_t *d_rec_offsets, int64_t n_records,
                  void *d_ids_out, int64_t ids_capacity, int64_t *d_out_offsets, void *stream);

/*
 * dnatok_pad: step 6.  Row r of d_batch_ids [n_records][seq_len] (int32) gets record r's first
 * min(tokens, seq_len) ids, LEFT: right-aligned, RIGHT: left-aligned; other columns pad_id.
 * d_mask [n_records][seq_len] (uint8) is 1 exactly on the kept columns; may be NULL.
 * d_ids / d_out_offsets are dnatok_encode's outputs (element type id_dtype).  Enqueue only.
 */
int dnatok_pad(dnatok_t *h, const void *d_ids, const int64_t *d_out_offsets, int64_t n_records,
               int32_t *d_batch_ids, uint8_t *d_mask, void *stream);

/*
 * dnatok_encode_pad: steps 1-6 in one call (PAPER.md:84 bytes path through PAPER.md:124-129 padding): d_out_offsets,
 * d_batch_ids and d_mask end up exactly as after dnatok_encode followed by dnatok_pad with the same arguments.  Inputs laid
 * out as wrapped FASTA or one line per record (see dnatok_set_fast_path) have their tokens written straight into the batch:
 * the CSR ids never travel through HBM, and d_ids_out is then left untouched.  Any other input is encoded into d_ids_out and
 * padded from there.  So d_ids_out / ids_capacity must be given as for dnatok_encode (workspace for the second case), but
 * the caller may rely on its contents only after dnatok_encode.  EINVAL if the handle has seq_len == 0.  Enqueue only.
 */
int dnatok_encode_pad(dnatok_t *h, const uint8_t *d_bytes, int64_t n_bytes, const int64_t *d_rec_offsets,
                      int64_t n_records, void *d_ids_out, int64_t ids_capacity, int64_t *d_out_offsets,
                      int32_t *d_batch_ids, uint8_t *d_mask, void *stream);

/* One delivered batch of dnatok_stream_encode (device pointers valid until the callback's stream work ends). */
typedef struct {
    int64_t first_record;        /* index of the first record in this batch                     */
    int64_t n_records;           /* records that END in this chunk (Q17), in order              */
    const void    *d_ids;        /* CSR ids (id_dtype) of these records                         */
    const int64_t *d_out_offsets;/* [n_records+1], relative to this batch                       */
    const int32_t *d_batch_ids;  /* [n_records][seq_len] or NULL when seq_len == 0              */
    const uint8_t *d_mask;       /* [n_records][seq_len] or NULL when seq_len == 0              */
    int64_t chunk_index;
    void   *stream;              /* cudaStream_t the batch was produced on                      */
} dnatok_batch;

typedef void (*dnatok_batch_fn)(void *user, const dnatok_batch *batch);

/*
 * dnatok_stream_encode: step 7.  Splits the host buffer into chunk_bytes pieces; chunk i goes to
 * device slot i mod n_streams on its own stream: H2D copy, carry of the record cut by the previous chunk
 * boundary, steps 1-6.  H2D of chunk i+1 overlaps the encode of chunk i.  Output equals dnatok_encode
 * (+ dnatok_pad) on the whole buffer, delivered batch by batch in record order; a record is delivered in
 * the chunk where it ends.  on_batch is called on the calling thread right after the batch's work has been
 * enqueued on batch->stream (enqueue consumer work there; the slot is recycled n_streams chunks later,
 * after that stream's work).  Returns after the last chunk has completed.
 *   h_bytes        [n_bytes] host memory.  Page-locked (cudaHostAlloc / cudaHostRegister / torch pin_memory): the
 *                  copies read it in place.  Pageable: every chunk is first copied into one of n_streams + 1 pinned
 *                  staging slots the handle owns (PAPER.md:181 persistent pinned buffers), at memcpy speed.
 *   h_rec_offsets  [n_records+1] host int64, same contract as dnatok_encode
 *   max_rows_per_chunk  upper bound on records ending in one chunk (sizes the per-slot batch tensors);
 *                  0 => chunk_bytes / 64 + 2.  Exceeding it returns DNATOK_ECAPACITY.
 * A record longer than cfg.max_record_bytes + chunk_bytes returns DNATOK_ECAPACITY.
 */
int dnatok_stream_encode(dnatok_t *h, const uint8_t *h_bytes, int64_t n_bytes,
                         const int64_t *h_rec_offsets, int64_t n_records,
                         int64_t chunk_bytes, int n_streams, int64_t max_rows_per_chunk,
                         dnatok_batch_fn on_batch, void *user);

/*
 * dnatok_stream_encode_from: the same with a PRODUCER instead of a buffer (a file reader, a decompressor).  For chunk i
 * the library calls fill(fill_user, i, offset, n, dst) on the calling thread; it must write bytes [offset, offset + n)
 * of the input to dst, a pinned staging slot (n_streams + 1 of them, so the producer of chunk i + 1 runs while the
 * copies and kernels of chunks i, i - 1, ... are in flight), and return 0; any other value aborts with EINVAL.
 * h_rec_offsets as above (known up front, e.g. from a .fai index).
 * On any failure of either call the ring's streams are drained before the call returns.
 */
typedef int (*dnatok_fill_fn)(void *fill_user, int64_t chunk_index, int64_t offset, int64_t n_bytes, uint8_t *dst);
int dnatok_stream_encode_from(dnatok_t *h, dnatok_fill_fn fill, void *fill_user, int64_t n_bytes,
                              const int64_t *h_rec_offsets, int64_t n_records,
                              int64_t chunk_bytes, int n_streams, int64_t max_rows_per_chunk,
                              dnatok_batch_fn on_batch, void *user);

/* Synchronise `stream` and report the handle's device status word: DNATOK_OK, DNATOK_ECAPACITY or
 * DNATOK_ESTATE (sticky until read).                                                                  */
int dnatok_check(dnatok_t *h, void *stream);

/* Message for the last non-OK return on this handle (never NULL; valid until the next call on h).      */
const char *dnatok_last_error(const dnatok_t *h);

/* ---------------------------------------------------------------------------------------------------------
 * operations next to the encoder.  All only enqueue on `stream`; none synchronises.
 * --------------------------------------------------------------------------------------------------------- */

/*
 * dnatok_revcomp (section 4.5.4: reverse complement on device).  Record r of d_out gets record
 * r of d_bytes reversed and complemented byte by byte: A<->T, C<->G, U->A, IUPAC R<->Y, K<->M, B<->V, D<->H;
 * S, W, N and every other byte (line breaks included) map to themselves; case is kept.  Bytes outside every
 * record are copied.  Meant for newline-free records (reverse complement, then dnatok_encode); d_out != d_bytes.
 * Same d_rec_offsets contract as dnatok_encode.
 */
int dnatok_revcomp(dnatok_t *h, const uint8_t *d_bytes, int64_t n_bytes, const int64_t *d_rec_offsets,
                   int64_t n_records, uint8_t *d_out, void *stream);

/*
 * dnatok_decode (section 4.5.2: decoding through an inverse vocabulary table).  Token ids of
 * dnatok_encode / rows of dnatok_pad (CSR: d_ids of id_dtype, d_out_offsets [n_records+1]) -> upper-case bases:
 *   single-nt: nt_ids[c] -> "ACGTN"[c], any other id -> 'N';  k-mer: base_id + code -> its k bases (first base most
 *   significant), base_id + 4^k + c -> "ACGTN"[c], any other id (UNK) -> k x 'N';  BPE: n_id -> 'N', base_id + t ->
 *   the spelling of token t, any other id -> 'N'.  pad_id tokens are skipped.
 * d_byte_offsets [n_records+1] int64 gets the exclusive prefix sum of the decoded record lengths; d_bytes_out
 * [bytes_capacity] the bytes (overflow: nothing written past the end, dnatok_check() returns DNATOK_ECAPACITY).
 * decode(encode(x)) == upper(stripped x) whenever x holds no N and no non-DNA byte.  EINVAL on a BPE handle whose
 * token spellings add up to more than 64 MiB.
 */
int dnatok_decode(dnatok_t *h, const void *d_ids, const int64_t *d_out_offsets, int64_t n_records,
                  uint8_t *d_bytes_out, int64_t bytes_capacity, int64_t *d_byte_offsets, void *stream);

/*
 * dnatok_decode_static: dnatok_decode for callers that may not allocate device memory (code under CUDA graph capture,
 * tight serving loops, harnesses that forbid cudaMalloc).  Same arguments, same results, but the call allocates and frees
 * NOTHING: its only scratch, the decoded length of every record, lives in a static device array inside the library of
 * DNATOK_DECODE_STATIC_MAX_RECORDS int32 (4 MiB, held by every GPU that loads the library until the process exits).
 * n_records beyond that maximum: DNATOK_ECAPACITY, nothing launched (use dnatok_decode, or split the records over calls).
 * Every handle and every call on a GPU shares the one array: calls that may overlap on the GPU (different streams, no
 * ordering between them) race on it -- order them, or use dnatok_decode, whose scratch belongs to the handle.  Nothing in
 * the array has to be cleared between calls (each call writes every entry it reads).  Enqueue only.
 */
#define DNATOK_DECODE_STATIC_MAX_RECORDS 1048576
int dnatok_decode_static(dnatok_t *h, const void *d_ids, const int64_t *d_out_offsets, int64_t n_records,
                         uint8_t *d_bytes_out, int64_t bytes_capacity, int64_t *d_byte_offsets, void *stream);

/* Rows per embedding call, PAPER.md:136 (Alg. 2 l.17) / PAPER.md:181: b = min(B_emb, max(1, floor(M / T'))).   */
int64_t dnatok_microbatch_rows(int64_t b_emb, int64_t m_tokens, int64_t t_len);

/* Called after the gather of rows [first_row, first_row + n_rows) has been enqueued on `stream`.               */
typedef void (*dnatok_microbatch_fn)(void *user, int64_t first_row, int64_t n_rows, void *d_out_rows, void *stream);

/*
 * dnatok_embed (PAPER.md:66-72 notation IDs [B x T'] -> [B x T' x D]; Alg. 2 l.18-24 micro-batch
 * loop): d_out[r][t][:] = d_table[d_ids[r][t]][:], rows of row_bytes bytes (D x element size; a multiple of 4,
 * 16-byte accesses when it and both pointers are multiples of 16); an id outside [0, vocab) gives a zero row.
 * The n_rows x t_len id matrix (int32, e.g. dnatok_pad's batch_ids) is processed dnatok_microbatch_rows(b_emb,
 * m_tokens, t_len) rows per launch, in order; on_microbatch (may be NULL) is called once per launch.  d_out holds
 * all n_rows x t_len x row_bytes bytes.
 */
int dnatok_embed(dnatok_t *h, const int32_t *d_ids, int64_t n_rows, int64_t t_len, const void *d_table,
                 int64_t vocab, int64_t row_bytes, void *d_out, int64_t b_emb, int64_t m_tokens,
                 dnatok_microbatch_fn on_microbatch, void *user, void *stream);

/* dnatok_widen_ids (IDs path "32-bit + on-device cast"): d_out[i] = (int64) d_ids[i], i < n.       */
int dnatok_widen_ids(dnatok_t *h, const int32_t *d_ids, int64_t n, int64_t *d_out, void *stream);

/* Number of kernels this library has launched on the handle since create (bench.py's gpu_launches).    */
int64_t dnatok_launch_count(const dnatok_t *h);

/*
 * Tuning knob of the single-pass encoder: the flat byte buffer is cut into super-tiles of
 * sub_tiles x 16 KiB, the unit of the chained scan.  0 (default) = chosen per call from n_bytes and the SM
 * count; 1..4 = fixed (tests use this to exercise every size on small inputs).  Results never depend on it.
 * EINVAL outside 0..4.
 */
int dnatok_set_super_tile(dnatok_t *h, int32_t sub_tiles);

/*
 * Test / tuning knob of the strip path: 1 (default) = inputs of 48 MiB or more go to the closed-form
 * encoder first, which assumes records laid out as an optional '>' header line followed by lines of one fixed width and
 * checks that layout on every byte; the chained-scan encoder runs behind it only if the check failed somewhere.  2 = the
 * same for inputs of any size (tests), 0 = the chained-scan encoder only.  Results never depend on it.  EINVAL outside 0..2.
 * With 1, two host-side rules keep hopeless attempts away: an input that averages more than 8 records per 16 KiB goes to the
 * chained-scan encoder directly, and after a call whose check failed (it then cost both encoders' time) the next 8 eligible
 * calls on the handle do too; the failure is read from a host-mapped word without synchronising, so it may take effect a
 * call or two late.
 */
int dnatok_set_fast_path(dnatok_t *h, int32_t enable);

/*
 * Synchronises `stream`, then says how the last dnatok_encode call on the handle was served: 1 = by the closed-form
 * encoder alone (the layout check held on every byte), 0 = by the chained-scan encoder (check failed, fast path off or
 * input under the size threshold, or another mode).  Negative = DNATOK_E*.  Tests use it to tell the two apart.
 */
int dnatok_fast_path_taken(dnatok_t *h, void *stream);

/*
 * Tuning / test knob: cap on the number of persistent CTAs the encode, BPE and pad kernels launch (0 = the
 * default, one grid's worth of resident CTAs).  Tests set 1, 2, 7 so that one CTA walks many super-tiles /
 * reads and every buffer-reuse path of the persistent kernels runs deterministically on small inputs.
 * Results never depend on it.  EINVAL if max_ctas < 0.
 */
int dnatok_set_grid_cap(dnatok_t *h, int32_t max_ctas);

/* Library version string, e.g. "dnatok-b200 0.1 (sm_100a)".                                            */
const char *dnatok_version(void);

#ifdef __cplusplus
}
#endif
#endif /* DNATOK_H */
