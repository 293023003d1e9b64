// Host planner of libmsa: descriptor validation, virtual-block flattening, causal horizons,
// persistent schedule with split-KV.  Pure host C++ (no CUDA calls) so it is testable on CPU.
#pragma once
#include <stdint.h>

#include <vector>

#include "../../include/msa.h"
#include "msa_plan.h"

namespace msa {

struct PlannerConfig {
    int Hq = 0, Hkv = 0, D = 0, G = 0;
    int R = 0;                  // tokens per 128-row tile: (128 / G) rounded down to a multiple of 8
    int tiles_per_group = 1;    // q tiles one work item covers (1 or 2)
    int num_ctas = 148;         // persistent CTAs available (SM count)
    int min_tiles_per_cta = 2;  // do not spread tiny problems thinner than this
    int snap_tiles = 2;         // a cut closer than this to an item boundary snaps onto it
};

struct HostPlan {
    std::vector<VBlock> vblocks;
    std::vector<WorkUnit> units;
    std::vector<int32_t> cta_unit_begin;   // [num_ctas_used + 1]
    std::vector<MergeItem> merge_items;
    std::vector<TileInfo> tile_info;
    std::vector<int32_t> vb_dst;           // write-back plans: per virtual block, block-table index of its destination or -1
    std::vector<int32_t> tile_writer;      // write-back plans: per context KV tile, q_row0 of the item that stores it or -1
    msa_plan_info info{};
    int64_t workspace_floats = 0;
    bool uses_paged = false, uses_contig = false;
    bool has_writeback = false;
    int64_t wb_max_bt = -1;                // largest block-table index a write-back job touches
};

// Returns MSA_OK or a negative MSA_ERR_* code.
// jobs / n_jobs: optional KV write-back fused into the forward launch (msa_plan_create_writeback).
int build_plan(const PlannerConfig &cfg, const msa_request *req, int32_t n_req, const msa_segment *seg, int32_t n_seg,
               HostPlan *out, const msa_append *jobs = nullptr, int32_t n_jobs = 0);

}  // namespace msa
