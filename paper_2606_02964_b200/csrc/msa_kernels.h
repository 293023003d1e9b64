// Launch interface between the host API (msa_api.cu) and the sm_100a kernels.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "msa_plan.h"

namespace msa {

struct FwdParams {
    CUtensorMap tm_q;        // bf16 [total_q][Hq*D], box 64 x R
    CUtensorMap tm_q3;       // the same tensor as [total_q][Hq][D], box 64 x G x R (token-major row packing, see token_major)
    // K/V tensors: pool bf16 [num_blocks*16][Hkv*D], arena bf16 [contig_rows][Hkv*D]; boxes of
    // 64 elements x {16, 8, 4, 2, 1} rows: a partly filled block loads only its valid rows.
    // fp8 pool: tm_pool_* are over bytes [num_blocks*16][Hkv*D] with boxes of D bytes x {16, 8, 4, 2, 1} rows, no swizzle.
    CUtensorMap tm_pool_k[5];
    CUtensorMap tm_ctg_k[5];
    CUtensorMap tm_pool_v[5];
    CUtensorMap tm_ctg_v[5];
    CUtensorMap tm_ctg_k128, tm_ctg_v128;   // arena, box 64 x 128: eight full consecutive blocks at once
    const VBlock *vblocks;
    const WorkUnit *units;
    const int32_t *cta_unit_begin;   // [num_ctas+1]
    const TileInfo *tile_info;
    const int32_t *block_table;
    const int32_t *vb_dst;           // fused KV write-back (NULL: none): per virtual block, block-table index of its destination or -1
    const int32_t *tile_writer;      // ... and per context KV tile, q_row0 of the work item that stores it (or -1)
    const int32_t *kv_to_q;          // [Hkv][G] q heads of each kv head
    const uint32_t *kv8_mul;         // fp8 pool only: [2][Hkv] f16 bits of 2^k for K then V, scale = 2^k (see e4m3x2_to_bf16x2)
    void *o;                         // bf16 [total_q][Hq][D]
    float *lse;                      // [total_q][Hq]
    float *workspace;
    float scale_log2;                // softmax_scale * log2(e)
    int32_t Hq, Hkv, G, R;           // R = tokens per 128-row tile
    int32_t token_major;             // 1: row r of a q tile = (token r / G, head r % G) -- the valid rows of a short query are
                                     // a prefix of the tile, so whole softmax warps have nothing to do; needs the q heads of
                                     // every KV head to be consecutive (one 3-D box loads a tile).  0: r = (head r / R, token r % R)
};

struct MergeParams {
    const MergeItem *items;
    const int32_t *kv_to_q;
    const float *workspace;
    void *o;
    float *lse;
    int32_t Hq, G, D;
};

// KV write-back: one unit = up to 16 tokens of one job
struct AppendUnit {
    int64_t src_row;       // first arena row
    int32_t bt_index;      // index into block_table of the destination block
    int32_t nvalid;        // tokens to copy, 1..16 (slots 0..nvalid-1 of the block)
};

struct AppendParams {
    const AppendUnit *units;
    const int32_t *block_table;
    const void *contig_k, *contig_v;
    void *pool_k, *pool_v;
    int64_t row_bytes;     // Hkv * D * 2 (arena row)
    int32_t n_units;
    const float *inv_scale; // fp8 pool: [2][Hkv] 1 / scale for K then V (the rows are quantised to E4M3); NULL for a bf16 pool
    int32_t Hkv, D;
};

// fp8 pool, dequantising pre-pass (msa_dequant.cu): block j of the bf16 copy = pool block block_table[src_bt[j]]
struct DequantParams {
    const int32_t *src_bt;        // [n_blocks] block-table indices, distinct
    const int32_t *block_table;
    const void *pool_k, *pool_v;  // E4M3 codes [num_blocks][16][Hkv][D]
    void *out_k, *out_v;          // bf16 [n_blocks][16][Hkv][D]
    int32_t *ident;               // [n_blocks], written 0, 1, 2, ...: the block table of the copy
    const uint32_t *kv8_mul;      // as in FwdParams
    int32_t n_blocks, Hkv, D;
};
cudaError_t launch_dequant(const DequantParams &p, int num_sms, cudaStream_t stream);

// Block-id check (msa_check.cu): entries of the block table a plan refers to
struct CheckParams {
    const VBlock *vblocks;        // forward plan: its virtual blocks (paged entries name a block-table index), or NULL
    const int32_t *vb_dst;        // write-back plan: destination block-table index per virtual block or -1, or NULL
    const AppendUnit *units;      // append plan: its copy units, or NULL
    int32_t n_vblocks, n_vb_dst, n_units;
    const int32_t *block_table;
    int64_t num_blocks;
    int32_t *flag;                // device int32: smallest offending block-table index, or -1
};
cudaError_t launch_check_ids(const CheckParams &p, bool reset, cudaStream_t stream);

cudaError_t configure_append();   // per device, like configure_fwd
cudaError_t launch_append(const AppendParams &p, int num_sms, cudaStream_t stream);

// Forward kernel: persistent, warp-specialised (msa_fwd_pipe.cuh).  configure_fwd sets the kernel's dynamic
// shared-memory limit on the CURRENT device (once per device and head dim); launch_fwd assumes it was done.
constexpr int kTilesPerGroup = 2;    // q tiles (of 128 packed rows) one work item covers in pair mode
cudaError_t configure_fwd(int head_dim, bool kv8);
// kv8: the pool tensor maps are over E4M3 codes (the fp8 variant converts them); one_q_tile: the plan has no pair-mode unit
cudaError_t launch_fwd(const FwdParams &p, int head_dim, bool kv8, bool one_q_tile, int num_ctas, cudaStream_t stream);
cudaError_t launch_merge(const MergeParams &p, int n_items, int max_rows, cudaStream_t stream);

}  // namespace msa
