// Host planner of libmsa (see msa_planner.h).  Turns the C-ABI descriptors into the device
// plan: the paper's "split indices" + per-token-block "equivalent seq_len" metadata
// (PAPER.md:122-124), re-designed as a virtual block list plus a persistent, split-KV
// schedule over (run, kv-head, q-tile, kv-tile-range) units.
#include "msa_planner.h"

#include <algorithm>
#include <climits>
#include <map>
#include <utility>

namespace msa {

namespace {

struct Ctx {
    int32_t vb_begin = 0;
    int32_t vb_count = 0;      // real (unpadded) virtual blocks
    int32_t ti_begin = 0;      // first TileInfo of the context
};

struct Item {
    int32_t q_row0, n_tok, q_abs0, kvh, vb_begin, vb_count, n_tiles, mode, ti_begin;
    int32_t cost;              // schedule cost of one KV tile of this item
};

// sum_{i=0}^{T-1} clamp(c0 + i, 0, n)
int64_t clamp_sum(int64_t c0, int64_t T, int64_t n)
{
    if (T <= 0 || n <= 0) return 0;
    const int64_t lo = c0, hi = c0 + T - 1;
    int64_t s = 0;
    const int64_t first = std::max<int64_t>(lo, 1), last = std::min<int64_t>(hi, n);
    if (last >= first) s += (first + last) * (last - first + 1) / 2;
    if (hi > n) s += n * (hi - std::max<int64_t>(n, lo - 1));
    return s;
}

}  // namespace

int build_plan(const PlannerConfig &cfg, const msa_request *req, int32_t n_req, const msa_segment *seg, int32_t n_seg,
               HostPlan *out, const msa_append *jobs, int32_t n_jobs)
{
    if (!out || n_req < 0 || n_seg < 0 || (n_req > 0 && !req) || (n_seg > 0 && !seg)) return MSA_ERR_INVALID_ARG;
    if (n_jobs < 0 || (n_jobs > 0 && !jobs)) return MSA_ERR_INVALID_ARG;
    if (cfg.G < 1 || cfg.R < 8 || cfg.tiles_per_group < 1 || cfg.num_ctas < 1) return MSA_ERR_INVALID_ARG;
    HostPlan &hp = *out;
    hp = HostPlan();

    // ---- segments: per-descriptor checks --------------------------------------------
    int64_t max_bt = -1, max_row = -1, max_q = -1;
    for (int32_t s = 0; s < n_seg; ++s) {
        const msa_segment &sg = seg[s];
        if (sg.kind < MSA_SEG_PAGED || sg.kind > MSA_SEG_SELF) return MSA_ERR_INVALID_ARG;
        if (sg.len < 1 || sg.abs_start < 0) return MSA_ERR_INVALID_ARG;
        if (static_cast<int64_t>(sg.abs_start) + sg.len > INT32_MAX) return MSA_ERR_OUT_OF_RANGE;
        if (sg.kind == MSA_SEG_PAGED) {
            if (sg.block_off < 0) return MSA_ERR_OUT_OF_RANGE;
            const int64_t last = static_cast<int64_t>(sg.block_off) + (sg.len + kBlock - 1) / kBlock - 1;
            if (last > INT32_MAX) return MSA_ERR_OUT_OF_RANGE;
            max_bt = std::max(max_bt, last);
        } else {
            if (sg.row_off < 0) return MSA_ERR_OUT_OF_RANGE;
            const int64_t last = sg.row_off + sg.len - 1;
            if (last + kBlock > INT32_MAX) return MSA_ERR_OUT_OF_RANGE;   // TMA coordinates are int32
            max_row = std::max(max_row, last);
        }
    }

    // ---- requests: ranges, q-row overlap ---------------------------------------------
    std::vector<std::pair<int64_t, int64_t>> qspans;
    for (int32_t r = 0; r < n_req; ++r) {
        const msa_request &rq = req[r];
        if (rq.q_len < 0 || rq.q_row_start < 0 || rq.q_abs_start < 0) return MSA_ERR_INVALID_ARG;
        if (rq.seg_begin < 0 || rq.seg_count < 0 || static_cast<int64_t>(rq.seg_begin) + rq.seg_count > n_seg)
            return MSA_ERR_OUT_OF_RANGE;
        if (static_cast<int64_t>(rq.q_abs_start) + rq.q_len > INT32_MAX) return MSA_ERR_OUT_OF_RANGE;
        if (static_cast<int64_t>(rq.q_row_start) + rq.q_len > INT32_MAX) return MSA_ERR_OUT_OF_RANGE;
        if (rq.q_len > 0) {
            qspans.emplace_back(rq.q_row_start, static_cast<int64_t>(rq.q_row_start) + rq.q_len);
            max_q = std::max<int64_t>(max_q, static_cast<int64_t>(rq.q_row_start) + rq.q_len - 1);
        }
    }
    std::sort(qspans.begin(), qspans.end());
    for (size_t i = 1; i < qspans.size(); ++i)
        if (qspans[i].first < qspans[i - 1].second) return MSA_ERR_OVERLAP;

    // ---- contexts: order / overlap checks, virtual block lists -----------------------
    std::map<std::pair<int32_t, int32_t>, Ctx> ctxs;
    for (int32_t r = 0; r < n_req; ++r) {
        const auto key = std::make_pair(req[r].seg_begin, req[r].seg_count);
        if (ctxs.count(key)) continue;
        for (int32_t s = key.first + 1; s < key.first + key.second; ++s) {
            if (seg[s].abs_start <= seg[s - 1].abs_start) {
                // equal starts always overlap (len >= 1); a smaller start is an ordering error
                return seg[s].abs_start == seg[s - 1].abs_start ? MSA_ERR_OVERLAP : MSA_ERR_UNSORTED;
            }
            if (static_cast<int64_t>(seg[s - 1].abs_start) + seg[s - 1].len > seg[s].abs_start) return MSA_ERR_OVERLAP;
        }
        Ctx c;
        c.vb_begin = static_cast<int32_t>(hp.vblocks.size());
        for (int32_t s = key.first; s < key.first + key.second; ++s) {
            const msa_segment &sg = seg[s];
            const int nblk = (sg.len + kBlock - 1) / kBlock;
            for (int b = 0; b < nblk; ++b) {
                VBlock vb;
                vb.paged = (sg.kind == MSA_SEG_PAGED) ? 1 : 0;
                vb.src = vb.paged ? sg.block_off + b : static_cast<int32_t>(sg.row_off + static_cast<int64_t>(b) * kBlock);
                vb.abs_start = sg.abs_start + b * kBlock;
                vb.nvalid = std::min(kBlock, sg.len - b * kBlock);
                hp.vblocks.push_back(vb);
            }
            if (sg.kind == MSA_SEG_PAGED) hp.uses_paged = true; else hp.uses_contig = true;
        }
        c.vb_count = static_cast<int32_t>(hp.vblocks.size()) - c.vb_begin;
        while ((hp.vblocks.size() - c.vb_begin) % kVbPerTile != 0) hp.vblocks.push_back(VBlock{0, INT32_MAX, 0, 0});
        if (hp.vblocks.size() > static_cast<size_t>(INT32_MAX)) return MSA_ERR_OUT_OF_RANGE;
        c.ti_begin = static_cast<int32_t>(hp.tile_info.size());
        for (size_t t = c.vb_begin; t < hp.vblocks.size(); t += kVbPerTile) {
            TileInfo ti{-1, 0};
            for (int b = 0; b < kVbPerTile; ++b) {
                const VBlock &vb = hp.vblocks[t + b];
                if (vb.nvalid < kBlock) ti.ragged = 1;
                if (vb.nvalid > 0) ti.max_abs = std::max(ti.max_abs, vb.abs_start + vb.nvalid - 1);
            }
            hp.tile_info.push_back(ti);
        }
        ctxs[key] = c;
    }

    // ---- fused KV write-back: which virtual block goes to which block-table entry ------------
    // A job's 16-token copy units must coincide with virtual blocks of the arena (same first row, same number of
    // valid slots): then the unit that loads a K/V tile for the attention can store it into the cache as it is.
    struct WbUnit { int32_t bt_index, nvalid; bool used; };
    std::map<int64_t, WbUnit> wb_units;          // first arena row -> destination
    if (n_jobs > 0) {
        std::vector<std::pair<int64_t, int64_t>> spans;
        for (int32_t j = 0; j < n_jobs; ++j) {
            const msa_append &a = jobs[j];
            if (a.len < 1 || a.row_off < 0 || a.block_off < 0) return MSA_ERR_INVALID_ARG;
            const int nblk = (a.len + kBlock - 1) / kBlock;
            const int64_t last_bt = static_cast<int64_t>(a.block_off) + nblk - 1;
            if (last_bt > INT32_MAX || a.row_off + a.len - 1 > INT32_MAX) return MSA_ERR_OUT_OF_RANGE;
            spans.emplace_back(a.block_off, last_bt + 1);
            hp.wb_max_bt = std::max(hp.wb_max_bt, last_bt);
            for (int b = 0; b < nblk; ++b) {
                const int64_t row = a.row_off + static_cast<int64_t>(b) * kBlock;
                if (wb_units.count(row)) return MSA_ERR_OVERLAP;
                wb_units[row] = WbUnit{a.block_off + b, std::min(kBlock, a.len - b * kBlock), false};
            }
        }
        std::sort(spans.begin(), spans.end());
        for (size_t i = 1; i < spans.size(); ++i)
            if (spans[i].first < spans[i - 1].second) return MSA_ERR_OVERLAP;
        hp.vb_dst.assign(hp.vblocks.size(), -1);
        for (size_t v = 0; v < hp.vblocks.size(); ++v) {
            const VBlock &vb = hp.vblocks[v];
            if (vb.paged || vb.nvalid <= 0) continue;
            auto it = wb_units.find(vb.src);
            if (it == wb_units.end()) continue;
            if (it->second.nvalid != vb.nvalid) return MSA_ERR_UNSUPPORTED;      // job and segment cut the rows differently
            hp.vb_dst[v] = it->second.bt_index;
            it->second.used = true;
        }
        for (const auto &kv : wb_units)
            if (!kv.second.used) return MSA_ERR_UNSUPPORTED;                      // rows no segment of this batch holds
        hp.has_writeback = true;
    }

    // ---- work items: (run, kv head, q-tile group), horizon folded in ------------------
    // tiles_per_group == 2: groups of 2R tokens run as kModePair (two q tiles share each KV
    // tile); a remainder of <= R tokens (and every short run) runs as kModeSplit.
    std::vector<Item> items;
    int64_t pairs = 0;
    for (int32_t r = 0; r < n_req; ++r) {
        const msa_request &rq = req[r];
        if (rq.q_len == 0) continue;
        const Ctx &c = ctxs[std::make_pair(rq.seg_begin, rq.seg_count)];
        for (int32_t s = rq.seg_begin; s < rq.seg_begin + rq.seg_count; ++s)
            pairs += clamp_sum(static_cast<int64_t>(rq.q_abs_start) - seg[s].abs_start + 1, rq.q_len, seg[s].len);
        for (int kvh = 0; kvh < cfg.Hkv; ++kvh) {
            int32_t t0 = 0;
            while (t0 < rq.q_len) {
                Item it;
                const int32_t left = rq.q_len - t0;
                if (cfg.tiles_per_group >= 2 && left > cfg.R) {
                    it.mode = kModePair;
                    it.n_tok = std::min<int32_t>(2 * cfg.R, left);
                } else {
                    it.mode = cfg.tiles_per_group >= 2 ? kModeSplit : kModePair;
                    it.n_tok = std::min<int32_t>(cfg.R, left);
                }
                it.cost = (cfg.tiles_per_group >= 2 && it.mode == kModePair) ? 2 : 1;
                it.q_row0 = rq.q_row_start + t0;
                it.q_abs0 = rq.q_abs_start + t0;
                it.kvh = kvh;
                it.vb_begin = c.vb_begin;
                it.ti_begin = c.ti_begin;
                const int32_t p_max = it.q_abs0 + it.n_tok - 1;
                // virtual blocks are in ascending abs_start: count those starting at or before p_max
                const VBlock *b0 = hp.vblocks.data() + c.vb_begin;
                const VBlock *e0 = b0 + c.vb_count;
                const VBlock *ub = std::upper_bound(b0, e0, p_max, [](int32_t p, const VBlock &v) { return p < v.abs_start; });
                it.vb_count = static_cast<int32_t>(ub - b0);
                it.n_tiles = (it.vb_count + kVbPerTile - 1) / kVbPerTile;
                items.push_back(it);
                t0 += it.n_tok;
            }
        }
    }

    // ---- write-back: which item stores which KV tile --------------------------------------------------------
    // All q-tile groups (items) of the runs that share a context load the same K/V tiles; the tiles that hold blocks
    // with a destination are dealt out round-robin among the items whose causal horizon reaches them, so the extra
    // stores are spread evenly over the units (the same assignment for every kv head).
    std::vector<uint8_t> item_writes(items.size(), 0);
    if (hp.has_writeback) {
        hp.tile_writer.assign(hp.tile_info.size(), -1);
        std::map<int32_t, std::vector<size_t>> by_ctx;                            // vb_begin -> items of kv head 0, in q order
        for (size_t i = 0; i < items.size(); ++i)
            if (items[i].kvh == 0) by_ctx[items[i].vb_begin].push_back(i);
        std::map<std::pair<int32_t, int32_t>, uint8_t> writes;                    // (vb_begin, q_row0) -> writes something
        for (const auto &kv : ctxs) {
            const Ctx &c = kv.second;
            const std::vector<size_t> &its = by_ctx[c.vb_begin];
            const int32_t n_tiles = (c.vb_count + kVbPerTile - 1) / kVbPerTile;
            for (int32_t t = 0; t < n_tiles; ++t) {
                bool any = false;
                int32_t last_b = -1;
                for (int b = 0; b < kVbPerTile && t * kVbPerTile + b < c.vb_count; ++b)
                    if (hp.vb_dst[c.vb_begin + t * kVbPerTile + b] >= 0) {
                        any = true;
                        last_b = t * kVbPerTile + b;
                    }
                if (!any) continue;
                std::vector<size_t> cand;
                for (size_t i : its)
                    if (items[i].vb_count > last_b) cand.push_back(i);           // loads every destination block of the tile
                if (cand.empty()) return MSA_ERR_UNSUPPORTED;                    // a row no query of this batch attends to
                const Item &w = items[cand[static_cast<size_t>(t) % cand.size()]];
                hp.tile_writer[c.ti_begin + t] = w.q_row0;
                writes[std::make_pair(c.vb_begin, w.q_row0)] = 1;
            }
        }
        for (size_t i = 0; i < items.size(); ++i)
            item_writes[i] = writes.count(std::make_pair(items[i].vb_begin, items[i].q_row0)) ? 1 : 0;
    }

    // ---- persistent schedule ------------------------------------------------------------
    // Every CTA gets the same share of the global (cost-weighted) tile count.  Two passes:
    //  1. whole items, block by block (a block = the q-tile groups of one (run, kv head), which
    //     all stream the SAME K/V), heaviest blocks first, each member onto one of the currently
    //     least loaded CTAs.  Equal loads mean equal start times, so the members of a block walk
    //     their common K/V tiles at the same time on different SMs and all but one of them hit in
    //     L2 (the contiguous-share schedule this replaces ran them back to back on ONE SM, a full
    //     pass of every other SM's traffic apart: 5.7x the algorithmic DRAM bytes on cfg2).
    //  2. the items that fit nowhere whole are cut along KV, stream-K style, into the capacity
    //     that is left, in CTA order; only those items need the merge kernel.
    const int64_t n_items = static_cast<int64_t>(items.size());
    std::vector<int64_t> icost(n_items);
    int64_t W = 0;
    for (int64_t i = 0; i < n_items; ++i) {
        icost[i] = static_cast<int64_t>(std::max<int32_t>(items[i].n_tiles, 1)) * items[i].cost;
        W += icost[i];
    }
    struct Piece { int64_t item; int32_t tb, te; };
    int n_used = 0;
    std::vector<std::vector<Piece>> queue;
    std::vector<int32_t> pieces(n_items, 0);
    if (W > 0) {
        n_used = static_cast<int>(std::min<int64_t>(cfg.num_ctas, std::max<int64_t>(1, W / std::max(1, cfg.min_tiles_per_cta))));
        queue.resize(n_used);
        std::vector<int64_t> cap(n_used), load(n_used, 0);
        for (int c = 0; c < n_used; ++c) cap[c] = (W * (c + 1)) / n_used - (W * c) / n_used;
        // blocks of consecutive items that share (context, kv head)
        struct Block { int64_t b0, b1, cost; };
        std::vector<Block> blocks;
        for (int64_t i = 0; i < n_items;) {
            int64_t j = i;
            int64_t cst = 0;
            while (j < n_items && items[j].vb_begin == items[i].vb_begin && items[j].kvh == items[i].kvh &&
                   (j == i || items[j].q_row0 > items[j - 1].q_row0)) {
                cst += icost[j];
                ++j;
            }
            blocks.push_back(Block{i, j, cst});
            i = j;
        }
        std::stable_sort(blocks.begin(), blocks.end(), [](const Block &x, const Block &y) {
            return x.cost * (y.b1 - y.b0) > y.cost * (x.b1 - x.b0);          // mean member cost, descending
        });
        std::vector<int> order(n_used);
        std::vector<int64_t> leftover;
        for (const Block &bl : blocks) {
            for (int64_t m0 = bl.b0; m0 < bl.b1; m0 += n_used) {
                const int64_t k = std::min<int64_t>(bl.b1 - m0, n_used);
                for (int c = 0; c < n_used; ++c) order[c] = c;
                std::partial_sort(order.begin(), order.begin() + k, order.end(),
                                  [&](int x, int y) { return load[x] != load[y] ? load[x] < load[y] : x < y; });
                for (int64_t j = 0; j < k; ++j) {
                    const int64_t it = m0 + j;
                    const int c = order[j];
                    if (load[c] + icost[it] <= cap[c] + cfg.snap_tiles) {
                        queue[c].push_back(Piece{it, 0, std::max<int32_t>(items[it].n_tiles, 0)});
                        load[c] += icost[it];
                        pieces[it] = 1;
                    } else {
                        leftover.push_back(it);
                    }
                }
            }
        }
        std::sort(leftover.begin(), leftover.end());
        // pass 2: the leftover items form one sequence; CTA c takes the range whose cost matches
        // the room it has left (cuts at the nearest tile boundary; a cut closer than snap_tiles to
        // an item edge moves onto the edge)
        const int64_t n_left = static_cast<int64_t>(leftover.size());
        std::vector<int64_t> lstart(n_left + 1, 0);
        for (int64_t k = 0; k < n_left; ++k) lstart[k + 1] = lstart[k] + icost[leftover[k]];
        const int64_t Wl = lstart[n_left];
        if (Wl > 0) {
            std::vector<int64_t> room(n_used);
            int64_t room_sum = 0;
            for (int c = 0; c < n_used; ++c) {
                room[c] = std::max<int64_t>(0, cap[c] - load[c]);
                room_sum += room[c];
            }
            std::vector<int64_t> bound(n_used + 1, 0);
            int64_t acc = 0;
            for (int c = 0; c < n_used; ++c) {
                acc += room[c];
                bound[c + 1] = room_sum > 0 ? (Wl * acc) / room_sum : (c + 1 == n_used ? Wl : 0);
            }
            bound[n_used] = Wl;
            for (int c = 1; c < n_used; ++c) {
                const int64_t bnd = bound[c];
                if (bnd <= 0 || bnd >= Wl) continue;
                const int64_t k = std::upper_bound(lstart.begin(), lstart.end(), bnd) - lstart.begin() - 1;   // item holding bnd
                const int64_t cost = items[leftover[k]].cost;
                const int64_t n_i = std::max<int32_t>(items[leftover[k]].n_tiles, 1);
                int64_t tcut = (bnd - lstart[k] + cost / 2) / cost;          // nearest tile boundary inside the item
                if (tcut <= cfg.snap_tiles) tcut = 0;
                else if (n_i - tcut <= cfg.snap_tiles) tcut = n_i;
                bound[c] = lstart[k] + tcut * cost;
            }
            for (int c = 1; c <= n_used; ++c) bound[c] = std::max(bound[c], bound[c - 1]);
            // two cuts inside one item closer than the snap window: drop the later one (the CTA
            // between them had next to no room anyway)
            for (int c = 1; c < n_used; ++c) {
                const int64_t k0 = std::upper_bound(lstart.begin(), lstart.end(), bound[c - 1]) - lstart.begin() - 1;
                if (k0 >= n_left || bound[c] <= bound[c - 1] || bound[c] >= lstart[k0 + 1]) continue;
                if (bound[c] - bound[c - 1] <= cfg.snap_tiles * static_cast<int64_t>(items[leftover[k0]].cost)) bound[c] = bound[c - 1];
            }
            int64_t k = 0;
            for (int c = 0; c < n_used; ++c) {
                const int64_t lo = bound[c], hi = bound[c + 1];
                while (k < n_left && lstart[k + 1] <= lo) ++k;
                for (int64_t j = k; j < n_left && lstart[j] < hi; ++j) {
                    const int64_t a = std::max(lo, lstart[j]), b2 = std::min(hi, lstart[j + 1]);
                    if (b2 <= a) continue;
                    const Item &it = items[leftover[j]];
                    Piece pc{leftover[j], 0, 0};
                    if (it.n_tiles > 0) {
                        pc.tb = static_cast<int32_t>((a - lstart[j]) / it.cost);
                        pc.te = static_cast<int32_t>((b2 - lstart[j]) / it.cost);
                    }
                    queue[c].push_back(pc);
                    ++pieces[leftover[j]];
                }
            }
        }
    }

    std::vector<int64_t> item_first_off(n_items, -1);
    std::vector<int32_t> item_emitted(n_items, 0);
    int64_t ws = 0;
    for (int64_t i = 0; i < n_items; ++i) {
        if (pieces[i] > 1) {
            const int64_t rows = static_cast<int64_t>(items[i].n_tok) * cfg.G;
            const int64_t stride = (rows * (cfg.D + 1) + 3) / 4 * 4;
            MergeItem mi;
            mi.q_row0 = items[i].q_row0;
            mi.n_tok = items[i].n_tok;
            mi.kvh = items[i].kvh;
            mi.n_partials = pieces[i];
            mi.first_off = ws;
            mi.stride = stride;
            hp.merge_items.push_back(mi);
            item_first_off[i] = ws;
            ws += stride * pieces[i];
        }
    }
    if (ws > static_cast<int64_t>(INT32_MAX)) return MSA_ERR_OUT_OF_RANGE;   // partial_off is int32 (floats)

    hp.cta_unit_begin.assign(n_used + 1, 0);
    for (int c = 0; c < n_used; ++c) {
        hp.cta_unit_begin[c] = static_cast<int32_t>(hp.units.size());
        for (const Piece &pc : queue[c]) {
            const Item &it = items[pc.item];
            WorkUnit u{};
            u.q_row0 = it.q_row0;
            u.n_tok = it.n_tok;
            u.q_abs0 = it.q_abs0;
            u.kvh = it.kvh;
            u.vb_begin = it.vb_begin;
            u.vb_count = it.vb_count;
            u.mode = it.mode;
            u.tile_info_begin = it.ti_begin;
            u.tile_begin = pc.tb;
            u.tile_end = pc.te;
            u.writeback = item_writes[pc.item];
            if (pieces[pc.item] > 1) {
                const int64_t rows = static_cast<int64_t>(it.n_tok) * cfg.G;
                const int64_t stride = (rows * (cfg.D + 1) + 3) / 4 * 4;
                u.partial_off = static_cast<int32_t>(item_first_off[pc.item] + stride * item_emitted[pc.item]);
                ++item_emitted[pc.item];
            } else {
                u.partial_off = -1;
            }
            hp.units.push_back(u);
        }
    }
    hp.cta_unit_begin[n_used] = static_cast<int32_t>(hp.units.size());

    hp.workspace_floats = ws;
    hp.info.num_ctas = n_used;
    hp.info.num_items = static_cast<int32_t>(n_items);
    hp.info.num_units = static_cast<int32_t>(hp.units.size());
    hp.info.num_split_items = static_cast<int32_t>(hp.merge_items.size());
    int32_t n_part = 0;
    for (const MergeItem &mi : hp.merge_items) n_part += mi.n_partials;
    hp.info.num_partials = n_part;
    hp.info.rows_per_tile = cfg.R * cfg.G;
    int64_t kv_tiles = 0;
    for (const Item &it : items) kv_tiles += it.n_tiles;
    hp.info.kv_tiles = kv_tiles;
    hp.info.visible_pairs = pairs;
    hp.info.max_block_table_index = hp.uses_paged ? max_bt : -1;
    hp.info.max_contig_row = hp.uses_contig ? max_row : -1;
    hp.info.max_q_row = max_q;
    return MSA_OK;
}

}  // namespace msa
