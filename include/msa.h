/*
 * msa.h -- C ABI of the B200-native Multi-Segment Attention (MSA) library (libmsa.so).
 *
 * MSA (arxiv/paper_2606_02964, section 4.1) computes exact causal
 * attention for runs of query tokens against a logically contiguous KV context that is
 * physically split into several segments.  Definition of the result, per query row i of a
 * run (absolute position p_i = q_abs_start + i) and q head h (KV head kvh = map[h]):
 *
 *     keys    = every token j of every segment of the run's segment list, at absolute
 *               position a_j = seg.abs_start + (index of the token in its segment)
 *     visible = { j : a_j <= p_i }                       (causal by absolute position)
 *     s_j     = softmax_scale * <q[i][h][:], K_j[kvh][:]>
 *     LSE     = ln sum_{visible} exp(s_j)                (natural log)
 *     O[d]    = sum_{visible} exp(s_j - LSE) * V_j[kvh][d]
 *     no visible key  =>  O = 0, LSE = -inf
 *
 * This is Eq. (1) (A = QK^T/sqrt(d_k), O = softmax(A)V) applied the way
 * Eq. (2) states it for several runs: each run attends to everything
 * that precedes it, cached or recomputed (Eq. (4)'s l1,q1,l2,q2 layout);
 * "only the attention module requires the token dependency information" and
 * one launch serves "any number of non-contiguous cache segments" of many requests
 * (PAPER.md:124).  Precision: bf16 q/k/v, fp32 accumulation, bf16 O, fp32 LSE.
 *
 * All pointers named "device" are CUDA device pointers on the handle's device; all others
 * are host pointers.  The library never takes ownership of caller memory.  No torch types
 * appear here; PyTorch (or anything else) only supplies device memory and a cudaStream_t.
 * Every call returns an int status (MSA_OK == 0, errors negative); nothing throws or aborts.
 */
#ifndef MSA_H_
#define MSA_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define MSA_BLOCK_SIZE 16          /* tokens per paged KV block */
#define MSA_MAX_GROUP 16           /* max q heads per KV head */

enum {
    MSA_OK = 0,
    MSA_ERR_INVALID_ARG = -1,      /* NULL pointer, negative size, non-positive / non-finite scale */
    MSA_ERR_UNSUPPORTED = -2,      /* head_dim not in {64,128}, block_size != 16, Hq % Hkv != 0, G > 16,
                                      head map that does not give every KV head exactly G q heads, an fp8 pool
                                      scale that is not a power of two in [2^-14, 2^7] */
    MSA_ERR_OVERLAP = -3,          /* segments of one request overlap in absolute position, or two
                                      requests write the same q rows */
    MSA_ERR_UNSORTED = -4,         /* segments of one request not in ascending abs_start */
    MSA_ERR_OUT_OF_RANGE = -5,     /* descriptor refers outside the extents given to msa_forward */
    MSA_ERR_MISALIGNED = -6,       /* device pointer not 16-byte aligned */
    MSA_ERR_WORKSPACE = -7,        /* workspace NULL / too small */
    MSA_ERR_CUDA = -8,             /* a CUDA runtime / driver call failed (see msa_last_cuda_error) */
    MSA_ERR_NO_DEVICE = -9,        /* no CUDA device, or the device is not sm_100 */
    MSA_ERR_STATIC_WS = -10        /* msa_forward_static_ws: the plan needs more scratch than MSA_STATIC_WS_BYTES (or the
                                      device ordinal is beyond the 64 the built-in scratch is tracked for) */
};

/* Segment kinds (BASELINE.json north_star):
 *   PAGED  -- cached tokens in 16-token blocks of the pool, reached through block_table
 *   CONTIG -- a run just recomputed into the contiguous arena
 *   SELF   -- the current chunk's own K/V, also rows of the contiguous arena           */
enum { MSA_SEG_PAGED = 0, MSA_SEG_CONTIG = 1, MSA_SEG_SELF = 2 };

/* Storage format of the paged pool (the KV cache; its footprint is what limits how much context stays resident,
 * PAPER.md:22).  The arena (recomputed runs, own chunk) and q / o are always bf16.
 *   MSA_POOL_BF16      bf16 elements
 *   MSA_POOL_FP8_E4M3  one byte per element, OCP FP8 E4M3 (1 sign, 4 exponent bits with bias 7, 3 mantissa bits, no
 *                      infinity, S.1111.111 = NaN), and one scale per KV head for K and one for V:
 *                          K_j[kvh][d] = e4m3(pool_k byte) * k_scale[kvh],   V_j[kvh][d] = e4m3(pool_v byte) * v_scale[kvh]
 *                      The scales must be powers of two in [2^-14, 2^7] (as in the OCP MX formats): the dequantised
 *                      value is then exactly a bf16, and the kernels multiply exactly that value (converted on chip
 *                      to bf16, or to f16 with the scale applied outside the MMA): same tolerances as the bf16 pool.
 *                      The plan decides how a launch is served, invisibly in the results: a launch of short queries
 *                      reads every cached byte once and converts it inside the forward kernel; a launch with prefill
 *                      chunks, which loads a cached tile once per q-tile group, first dequantises the blocks it refers
 *                      to into the workspace, once, and runs the bf16 kernel on that copy (msa_workspace_bytes grows
 *                      accordingly).  The short-query launch multiplies in f16: code * 2^k is exact in f16 for every
 *                      legal scale, and q and the arena rows it meets are converted bf16 -> f16 as they are.  An fp8
 *                      handle therefore asks |q|, |arena K|, |arena V| <= 65504 whatever the scales are (larger magnitudes
 *                      saturate to +-65504; magnitudes below 2^-14 are rounded to a multiple of 2^-24).  A NaN code
 *                      dequantises to an unspecified value, possibly NaN (non-finite K/V are outside the definition,
 *                      DESIGN.md c19); codes in slots no query row can see never reach O. */
enum { MSA_POOL_BF16 = 0, MSA_POOL_FP8_E4M3 = 1 };

typedef struct {
    int32_t num_q_heads;           /* Hq                                                     */
    int32_t num_kv_heads;          /* Hkv, divides Hq; G = Hq/Hkv <= 16                      */
    int32_t head_dim;              /* D in {64, 128}                                         */
    int32_t block_size;            /* must be 16                                             */
    const int32_t *q_to_kv_head;   /* host int32[Hq] GQA head map, or NULL => h / G (Llama)  */
    int32_t device;                /* CUDA device ordinal                                    */
    int32_t pool_format;           /* MSA_POOL_BF16 (0) or MSA_POOL_FP8_E4M3                 */
    const float *k_scale;          /* fp8 pool: host fp32[Hkv] (copied); NULL => all 1.0     */
    const float *v_scale;          /* fp8 pool: host fp32[Hkv] (copied); NULL => all 1.0     */
} msa_config;

typedef struct {
    int32_t kind;                  /* MSA_SEG_*                                              */
    int32_t abs_start;             /* absolute position of the segment's first token, >= 0   */
    int32_t len;                   /* tokens, >= 1; the last paged block may be partly filled */
    int32_t block_off;             /* PAGED: index into block_table of the segment's first
                                      block; token idx lives in block block_table[block_off +
                                      idx/16], slot idx%16 (a PAGED segment starts at slot 0) */
    int64_t row_off;               /* CONTIG/SELF: arena row of the segment's first token     */
} msa_segment;

typedef struct {
    int32_t q_row_start;           /* first row of q / o / lse of this query run             */
    int32_t q_len;                 /* rows (tokens) of the run, >= 0                         */
    int32_t q_abs_start;           /* absolute position of the run's first token             */
    int32_t seg_begin, seg_count;  /* slice of the segment array this run attends to;
                                      several runs may share one slice (hybrid chunks,
                                      PAPER.md:92 step 5, :247).  Ascending abs_start, no
                                      overlap; gaps are legal (attention over the union).    */
} msa_request;

typedef struct {
    int32_t num_ctas;              /* persistent CTAs the forward kernel is launched with    */
    int32_t num_items;             /* (run, kv-head, q-tile) work items                      */
    int32_t num_units;             /* (item, kv-tile-range) units after split-KV             */
    int32_t num_split_items;       /* items whose KV range was split (need the merge kernel) */
    int32_t num_partials;          /* partial (O, LSE) results written to the workspace      */
    int32_t rows_per_tile;         /* packed (token, q-head) rows per 128-row MMA tile used  */
    int64_t kv_tiles;              /* total 128-key tiles visited                            */
    int64_t visible_pairs;         /* sum over rows of visible keys, per q head              */
    int64_t max_block_table_index; /* extents the plan needs at msa_forward                  */
    int64_t max_contig_row;
    int64_t max_q_row;
} msa_plan_info;

typedef struct msa_handle_s *msa_handle;
typedef struct msa_plan_s *msa_plan;

/*
 * Create a handle for one model shape on one device.  Owns only small host state and a
 * few KB of device memory.  Fails with MSA_ERR_NO_DEVICE when there is no sm_100 GPU:
 * there is no CPU fallback.  cfg->device < 0 makes a planning-only handle (descriptor
 * validation and scheduling on the host, for tools and tests); msa_forward on it returns
 * MSA_ERR_NO_DEVICE.
 */
int msa_create(const msa_config *cfg, msa_handle *out);
void msa_destroy(msa_handle h);

/* Build the launch plan for a batch of query runs (host arrays, copied; may be freed after
 * the call).  This is the paper's attention metadata -- "split indices" and the per-token-
 * block "equivalent seq_len" array -- plus the persistent tile schedule
 * and split-KV decisions.  All descriptor validation happens here.  The plan depends only
 * on lengths and residency, not on tensor values or block ids, so one plan serves every
 * layer of a model step.  Owns a small device buffer; uploads it synchronously. */
int msa_plan_create(msa_handle h, const msa_request *requests, int32_t n_req,
                    const msa_segment *segments, int32_t n_seg, msa_plan *out);
void msa_plan_destroy(msa_plan p);
int msa_plan_get_info(msa_plan p, msa_plan_info *info);

/* Introspection (tests, tools): copy one of the plan's host-side arrays out.
 *   which = 0  virtual blocks      int32[4]  {src, abs_start, nvalid, paged}
 *           1  work units          int32[12] {q_row0, n_tok, q_abs0, kvh, vb_begin, vb_count,
 *                                             tile_begin, tile_end, partial_off, mode,
 *                                             tile_info_begin, 0}
 *           2  cta_unit_begin      int32     [num_ctas + 1]
 *           3  merge items         {int32 q_row0, n_tok, kvh, n_partials; int64 first_off, stride}
 *           4  tile mask summaries int32[2]  {max_abs, ragged} per context KV tile
 *           7  fp8 pool: block-table indices the dequantising pre-pass converts (int32; empty when the forward kernel
 *              converts the codes itself)
 * With buf == NULL only *bytes is set; otherwise *bytes is the capacity on entry. */
int msa_plan_export(msa_plan p, int which, void *buf, size_t *bytes);

/* Bytes of device scratch msa_forward needs for this plan (split-KV partials; on an fp8 handle also the bf16 copy of the
 * cached blocks of a launch that loads them several times, see MSA_POOL_FP8_E4M3); may be 0. */
int msa_workspace_bytes(msa_plan p, size_t *bytes);

/* One MSA forward pass, asynchronous on `cuda_stream` (a cudaStream_t; NULL = default
 * stream).  Never allocates, never synchronises, never reads device memory on the host.
 * Calls on ONE handle (msa_forward*, msa_kv_append, msa_set/get_timing) must not run concurrently on
 * several host threads: the handle keeps the encoded tensor maps of the last 64 pointer sets and the
 * launch counter.  Different handles are independent.
 *
 *   q            device bf16 [total_q][Hq][D]
 *   pool_k/v     device bf16 [num_blocks][16][Hkv][D]      (paged KV cache; E4M3 bytes of the same shape when the
 *                                                          handle was created with MSA_POOL_FP8_E4M3)
 *   block_table  device int32 [block_table_len], physical block ids in logical order
 *   contig_k/v   device bf16 [contig_rows][Hkv][D]         (recomputed runs + own chunk)
 *   o            device bf16 [total_q][Hq][D]   (written for every row of every run)
 *   lse          device fp32 [total_q][Hq]      (natural log; -inf for rows with no key)
 *   workspace    device, >= msa_workspace_bytes(), 16-byte aligned; may be NULL if 0 bytes
 *
 * Rows of q/o/lse not covered by any run are left untouched.  pool/contig pointers may be
 * NULL when the plan references no segment of that kind.  Block ids are trusted (they live
 * on the device; msa_check_block_ids validates them on request); slots past a segment's length and unused blocks may hold anything,
 * including NaN: they never reach O. */
int msa_forward(msa_handle h, msa_plan p,
                const void *q, int64_t total_q,
                const void *pool_k, const void *pool_v, int64_t num_blocks,
                const int32_t *block_table, int64_t block_table_len,
                const void *contig_k, const void *contig_v, int64_t contig_rows,
                float softmax_scale,
                void *o, float *lse,
                void *workspace, size_t workspace_bytes, void *cuda_stream);

/* ---- msa_forward without a workspace argument: the scratch is built into the library ----
 * Who this is for.  msa_forward wants `workspace` bytes from the caller, and a caller normally gets them from cudaMalloc.
 * Two kinds of caller of this library cannot do that at step time:
 *   - a serving engine that sized its paged KV pool to whatever HBM was free at start-up (the pool's size is what decides
 *     how much context stays resident): nothing is left for cudaMalloc to hand out later, and the
 *     workspace size changes with every batch's split-KV schedule, so it cannot be sized once either;
 *   - code that runs while other streams have steps in flight and must not stall them: cudaMalloc and cudaFree
 *     synchronise the whole device, and some hosts (a plugin inside another framework's memory manager) are simply not
 *     allowed to call them.
 * For them the library carries MSA_STATIC_WS_BYTES of device memory of its own -- a fixed array inside libmsa.so's device
 * image -- and this call uses it as the workspace: split-KV partials written by the forward kernel and read by the LSE-merge
 * kernel, and on an fp8 handle the bf16 copy of the cached blocks a prefill launch dequantises first.
 *
 * Arguments, results and status codes are those of msa_forward (same kernels, bit-identical O / LSE), minus `workspace` /
 * `workspace_bytes`.  A plan whose msa_workspace_bytes() exceeds MSA_STATIC_WS_BYTES is refused with MSA_ERR_STATIC_WS and
 * nothing is launched (32 MiB covers every bf16-pool batch of BASELINE.json: the largest, cfg3, needs 26.7 MiB; an fp8
 * prefill plan that copies more than that much of the pool does not fit -- use msa_forward there).
 *
 * Cost: every GPU on which the array's module gets loaded gives up MSA_STATIC_WS_BYTES until the process exits, whether
 * or not this call is ever used again.
 *
 * The call itself allocates no device memory and frees none (no cudaMalloc / cudaFree / cudaMallocAsync, no library
 * routine that allocates; msa_create and msa_plan_create, which own small device buffers, are set-up calls and are not
 * covered by this promise).  The FIRST call on a device does a one-time set-up: it looks up the array's device address
 * (with the CUDA runtime's default lazy module loading this is also the moment that part of the library is loaded on the
 * device and the 32 MiB are actually reserved; with CUDA_MODULE_LOADING=EAGER that happens when the context is created).
 * Make that first call at start-up, on any small split-KV or ordinary plan, before the engine takes the rest of the
 * memory and before any stream capture is begun.
 *
 * Sharing: there is ONE array per device, shared by every handle, plan and thread of the process.  Two calls that may
 * run on the GPU at the same time (different streams, or different threads without ordering) overwrite each other's
 * partials: issue them on one stream, or order them with events.  The array keeps whatever the last call left in it.
 * Nothing in it has to start at zero -- every float the merge kernel reads was written by the forward kernel of the same
 * call, and the fp8 copy and its index table are rewritten in full by the pre-pass -- so the call clears nothing. */
#define MSA_STATIC_WS_BYTES (32u << 20)
int msa_forward_static_ws(msa_handle h, msa_plan p,
                          const void *q, int64_t total_q,
                          const void *pool_k, const void *pool_v, int64_t num_blocks,
                          const int32_t *block_table, int64_t block_table_len,
                          const void *contig_k, const void *contig_v, int64_t contig_rows,
                          float softmax_scale,
                          void *o, float *lse, void *cuda_stream);

/* End-to-end convenience call with HOST buffers for everything a serving step produces:
 * q, the block table, the contiguous arena (recomputed runs + own chunk) come from host
 * memory and O / LSE go back to host memory; the paged pool is the resident KV cache and
 * stays a device pointer.  Copies are issued on `cuda_stream` around the same kernels as
 * msa_forward, using staging buffers owned by the handle (grown on demand, so the first
 * call may allocate); the call returns after the results have landed (it synchronises the
 * stream).  Host buffers should be pinned for full PCIe speed but need not be.  All total_q
 * rows of o_host / lse_host are overwritten; rows not covered by any run hold unspecified
 * values. */
int msa_forward_host(msa_handle h, msa_plan p,
                     const void *q_host, int64_t total_q,
                     const void *pool_k, const void *pool_v, int64_t num_blocks,
                     const int32_t *block_table_host, int64_t block_table_len,
                     const void *contig_k_host, const void *contig_v_host, int64_t contig_rows,
                     float softmax_scale,
                     void *o_host, float *lse_host, void *cuda_stream);

/* The same call without the wait, for a caller that keeps two steps in flight: the uploads run on a stream of the handle's
 * own, the kernels on `cuda_stream`, the read-back on a second stream of the handle's, chained by events, and each of the
 * two `slot`s (0 or 1) has its own staging buffers -- so the upload of one call overlaps the kernels and the read-back of the
 * call before it (PCIe is full duplex).  o_host / lse_host of a call are valid after msa_forward_host_wait(h, slot) (or after
 * the next msa_forward_host_async on the same slot, which waits for it first); the host input buffers must stay unchanged
 * until then.  msa_forward_host = msa_forward_host_async on slot 0 + msa_forward_host_wait. */
int msa_forward_host_async(msa_handle h, msa_plan p,
                           const void *q_host, int64_t total_q,
                           const void *pool_k, const void *pool_v, int64_t num_blocks,
                           const int32_t *block_table_host, int64_t block_table_len,
                           const void *contig_k_host, const void *contig_v_host, int64_t contig_rows,
                           float softmax_scale,
                           void *o_host, float *lse_host, void *cuda_stream, int32_t slot);
int msa_forward_host_wait(msa_handle h, int32_t slot);

/* ---- KV write-back (PAPER.md:92 step 2: recomputed K/V are written into cache blocks) ----
 * After a step, the K/V rows a request has just (re)computed -- CONTIG and SELF segments of the arena -- are appended
 * to the paged cache so that the next step can reach them as PAGED segments.  One job copies arena rows
 * [row_off, row_off + len) into the blocks block_table[block_off + i/16], slot i%16 (the same addressing a PAGED
 * segment uses: the job starts at slot 0 of its first block; a partly filled last block leaves its tail untouched). */
typedef struct {
    int64_t row_off;               /* first arena row                                        */
    int32_t len;                   /* tokens, >= 1                                           */
    int32_t block_off;             /* index into block_table of the first destination block  */
} msa_append;

typedef struct msa_append_plan_s *msa_append_plan;

/* Validates the jobs (host array, copied) and uploads the 16-token copy units.  MSA_ERR_INVALID_ARG for a bad job,
 * MSA_ERR_OVERLAP if two jobs write the same block-table entry.  n_jobs = 0 is legal (msa_kv_append launches nothing). */
int msa_append_plan_create(msa_handle h, const msa_append *jobs, int32_t n_jobs, msa_append_plan *out);
void msa_append_plan_destroy(msa_append_plan ap);

/* Asynchronous on `cuda_stream`, one kernel launch; never allocates or synchronises.  contig_* / pool_* / block_table as
 * in msa_forward, except that the pool is written.  The destination blocks must not be read by a kernel running
 * concurrently on another stream.  MSA_ERR_OUT_OF_RANGE if a job exceeds contig_rows or block_table_len (block ids
 * themselves are trusted, they live on the device -- and here a bad id is a wild write: msa_check_block_ids checks them); MSA_ERR_MISALIGNED for pointers not 16-byte aligned. */
/* fp8 pool: the rows are quantised on the way, code = E4M3 code nearest to arena value / scale (ties to the even code,
 * |value / scale| > 448 saturates to +-448, NaN gives the NaN code), so that e4m3(code) * scale is what a later PAGED
 * segment reads. */
int msa_kv_append(msa_handle h, msa_append_plan ap,
                  const void *contig_k, const void *contig_v, int64_t contig_rows,
                  void *pool_k, void *pool_v, int64_t num_blocks,
                  const int32_t *block_table, int64_t block_table_len, void *cuda_stream);

/* ---- KV write-back fused into the forward launch ----
 * The forward kernel already brings every K/V row of a recomputed (CONTIG) or own (SELF) segment into shared memory;
 * with a write-back plan the unit that loads a tile for the attention also stores it into its cache blocks (one TMA
 * store per 16-token block and 64-element half, straight from the tile), so no second pass over the arena and no second
 * launch is needed (PAPER.md:92 step 2 "allocates cache blocks": in the paper's engine the recomputed K/V land in
 * paged blocks within the same step).
 *
 * msa_plan_create_writeback = msa_plan_create + `jobs` (same meaning as in msa_append_plan_create).  Restrictions, each
 * reported as MSA_ERR_UNSUPPORTED (use msa_kv_append then): every 16-token copy unit of a job must coincide with a
 * 16-token block of a CONTIG / SELF segment of the batch (same first arena row, same number of tokens), and some query
 * row of the batch must attend to it (a row nobody reads is never loaded).  MSA_ERR_OVERLAP / MSA_ERR_INVALID_ARG /
 * MSA_ERR_OUT_OF_RANGE as in msa_append_plan_create.  n_jobs = 0 gives an ordinary plan.
 *
 * msa_forward_writeback = msa_forward on such a plan, except that pool_k / pool_v are written: after the call has
 * completed on the stream, pool[block_table[job.block_off + i/16]][i%16] = arena[job.row_off + i] for every job, bit for
 * bit, and O / LSE are bit-identical to msa_forward on the same plan.  The destination blocks must not be read by this
 * or any concurrently running call.  MSA_ERR_INVALID_ARG if the plan has no write-back jobs; MSA_ERR_OUT_OF_RANGE if a
 * job's block-table slice exceeds block_table_len.  msa_forward on a write-back plan computes O / LSE only.
 *
 * fp8 pool: the same two calls work, but the store is not fused -- the forward kernel moves bf16 tiles as they are and cannot
 * quantise them -- so msa_forward_writeback issues the forward kernel and then msa_kv_append's quantising kernel on the
 * same stream (one more launch; the bytes written are those of msa_kv_append, O / LSE those of msa_forward).  The
 * restrictions on the jobs above do not apply there; the validation is msa_append_plan_create's. */
int msa_plan_create_writeback(msa_handle h, const msa_request *requests, int32_t n_req,
                              const msa_segment *segments, int32_t n_seg,
                              const msa_append *jobs, int32_t n_jobs, msa_plan *out);
int msa_forward_writeback(msa_handle h, msa_plan p,
                          const void *q, int64_t total_q,
                          void *pool_k, void *pool_v, int64_t num_blocks,
                          const int32_t *block_table, int64_t block_table_len,
                          const void *contig_k, const void *contig_v, int64_t contig_rows,
                          float softmax_scale,
                          void *o, float *lse,
                          void *workspace, size_t workspace_bytes, void *cuda_stream);

/* ---- Debug check of the block ids (ids live on the device and are validated only on request) ----
 * msa_forward, msa_forward_writeback and msa_kv_append trust the ids in block_table: the loads and the fused write-back go
 * through tensor maps, which clip a box that leaves the pool, but msa_kv_append forms global addresses from the ids, so a
 * bad id there is a wild write.  A caller that wants to be sure runs this first: one small kernel looks at exactly the
 * block-table entries the plan refers to (the PAGED segments of `p`, its write-back destinations, the jobs of `ap`; either
 * of p / ap may be NULL, not both) and leaves in *device_flag (device int32) the smallest block-table index whose id is
 * outside [0, num_blocks), or -1 if all are fine.  Entries the plan does not use are not looked at (they may hold stale
 * ids).  Asynchronous on `cuda_stream`: read the flag after the stream has caught up.  Never allocates or synchronises.
 * MSA_ERR_OUT_OF_RANGE if a plan needs more than block_table_len entries. */
int msa_check_block_ids(msa_handle h, msa_plan p, msa_append_plan ap,
                        const int32_t *block_table, int64_t block_table_len, int64_t num_blocks,
                        int32_t *device_flag, void *cuda_stream);

/* Number of kernels the last msa_forward / msa_forward_host on this handle launched. */
int msa_last_launch_count(msa_handle h);

/* Per-kernel device timing for benchmarks.  msa_set_timing(h, n) makes the next n calls of
 * msa_forward record CUDA events on their stream around the forward kernel and the merge
 * kernel (n = 0 switches it off); msa_get_timing waits for the last recorded step, returns
 * how many steps were recorded and the average duration of each kernel in milliseconds,
 * and restarts the recording window. */
int msa_set_timing(msa_handle h, int max_steps);
int msa_get_timing(msa_handle h, int32_t *steps, double *fwd_ms_avg, double *merge_ms_avg);

const char *msa_strerror(int status);
/* Text of the last CUDA error seen by this thread inside the library ("" if none). */
const char *msa_last_cuda_error(void);
const char *msa_version(void);

#ifdef __cplusplus
}
#endif
#endif /* MSA_H_ */
