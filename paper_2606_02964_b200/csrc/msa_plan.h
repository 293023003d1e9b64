// Internal plan layout of libmsa: what the host planner (msa_plan.cpp) uploads and the
// sm_100a kernels (msa_fwd.cu, msa_merge.cu) read.  Not part of the C ABI.
//
// The paper's kernel is told where segments start and how much KV each token block may
// see through "split indices" and a precomputed per-token-block "equivalent seq_len"
// array.  Here that metadata is:
//   * a per-context *virtual block list*: one 16-byte entry per <=16 consecutive tokens of
//     one segment, paged or contiguous alike, carrying where the rows live, the absolute
//     position of the first token and how many of the 16 slots are valid;
//   * work units (run, kv-head, q-tile, kv-tile-range): the persistent schedule, with the
//     causal horizon already folded into the tile range.
#pragma once
#include <stdint.h>

namespace msa {

constexpr int kBlock = 16;            // tokens per virtual block (== paged block size)
constexpr int kTileN = 128;           // keys per KV tile
constexpr int kVbPerTile = kTileN / kBlock;
constexpr int kTileM = 128;           // packed (head, token) rows per MMA tile

struct alignas(16) VBlock {
    int32_t src;        // paged: index into block_table; contiguous: first arena row
    int32_t abs_start;  // absolute position of slot 0 (INT32_MAX for padding entries)
    int32_t nvalid;     // valid slots, 1..16 (0 for padding entries)
    int32_t paged;      // 1 = paged pool (row = block_table[src]*16), 0 = contiguous arena
};
// Every context's list is padded with {0, INT32_MAX, 0, 0} entries to a multiple of 8, so a
// KV tile always has 8 readable entries.

// One unit = one q-tile group of one (run, kv head) against a contiguous range of KV tiles.
struct alignas(16) WorkUnit {
    int32_t q_row0;        // global q row of the group's first token
    int32_t n_tok;         // valid tokens in the group (<= tiles_per_group * R)
    int32_t q_abs0;        // absolute position of the first token
    int32_t kvh;           // kv head
    int32_t vb_begin;      // first virtual block of the run's context
    int32_t vb_count;      // virtual blocks inside the group's causal horizon
    int32_t tile_begin;    // KV tiles [tile_begin, tile_end) of 8 virtual blocks each
    int32_t tile_end;
    int32_t partial_off;   // < 0: writes final O/LSE; else float offset of this unit's partial
    int32_t mode;          // kModePair: two q tiles share every KV tile (prefill chunks);
                           // kModeSplit: one q tile, even/odd KV tiles go to the two softmax
                           // warpgroups and are merged in the epilogue (short queries)
    int32_t tile_info_begin;  // index of the context's first TileInfo
    int32_t writeback;        // 1: this unit stores some of the K/V tiles it loads into the paged cache (HostPlan::tile_writer, vb_dst)
};

constexpr int kModePair = 0;
constexpr int kModeSplit = 1;

// Per context KV tile: what the softmax warps need to decide whether a tile needs masking.
struct alignas(8) TileInfo {
    int32_t max_abs;       // largest absolute position of a valid slot in the tile (-1 if none)
    int32_t ragged;        // 1 if any of the 8 virtual blocks has fewer than 16 valid slots
};

// Items whose KV range was split: the merge kernel combines their partials in tile order.
struct alignas(16) MergeItem {
    int32_t q_row0;
    int32_t n_tok;
    int32_t kvh;
    int32_t n_partials;
    int64_t first_off;     // float offset of partial 0; partial s at first_off + s*stride
    int64_t stride;        // floats per partial = round_up(rows*(D+1), 4), rows = n_tok*G
};

// Partial layout (floats): O_part[rows][D] (normalised), then LSE_part[rows]; row = g*n_tok + t.

}  // namespace msa
