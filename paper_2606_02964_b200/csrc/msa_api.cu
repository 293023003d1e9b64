// C ABI of libmsa (include/msa.h): handle, plan upload, tensor-map encoding and launches.
#include <cuda.h>
#include <limits.h>
#include <cuda_runtime.h>
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <algorithm>
#include <mutex>
#include <new>
#include <string>
#include <vector>

#include "../../include/msa.h"
#include "msa_kernels.h"
#include "msa_planner.h"

using namespace msa;

namespace {

thread_local std::string g_cuda_err;

int cuda_fail(cudaError_t e, const char *what)
{
    g_cuda_err = std::string(what) + ": " + cudaGetErrorString(e);
    cudaGetLastError();
    return MSA_ERR_CUDA;
}
#define MSA_CUDA(expr)                                         \
    do {                                                       \
        cudaError_t e_ = (expr);                               \
        if (e_ != cudaSuccess) return cuda_fail(e_, #expr);    \
    } while (0)

typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                  const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

// Makes the handle's device current for the duration of a call and restores the caller's afterwards.
struct DeviceGuard {
    int prev = -1;
    cudaError_t err = cudaSuccess;
    explicit DeviceGuard(int device)
    {
        err = cudaGetDevice(&prev);
        if (err == cudaSuccess && prev != device) err = cudaSetDevice(device);
        else if (err == cudaSuccess) prev = -1;       // nothing to restore
    }
    ~DeviceGuard()
    {
        if (prev >= 0) cudaSetDevice(prev);
    }
};

struct DevBuf {
    void *p = nullptr;
    size_t cap = 0;
    cudaError_t reserve(size_t bytes)
    {
        if (bytes <= cap) return cudaSuccess;
        if (p) cudaFree(p);
        p = nullptr;
        cap = 0;
        cudaError_t e = cudaMalloc(&p, bytes);
        if (e == cudaSuccess) cap = bytes;
        return e;
    }
    void release()
    {
        if (p) cudaFree(p);
        p = nullptr;
        cap = 0;
    }
};

}  // namespace

constexpr size_t kMapCacheEntries = 64;

struct msa_handle_s {
    msa_config cfg{};
    int G = 0, R = 0;
    int num_sms = 0;
    bool planning_only = false;
    std::vector<int32_t> kv_to_q;      // [Hkv][G]
    int32_t *d_kv_to_q = nullptr;
    bool token_major = false;          // q heads of every KV head are consecutive: q tiles are packed token-major (FwdParams::token_major)
    bool kv8 = false;                  // fp8 (E4M3) paged pool
    std::vector<float> kv_scale;       // kv8: [2][Hkv] K scales then V scales (powers of two)
    uint32_t *d_kv8_mul = nullptr;     // kv8: [2][Hkv] f16 bits of 2^k (forward kernel)
    float *d_kv8_inv = nullptr;        // kv8: [2][Hkv] 1 / scale (quantising msa_kv_append)
    EncodeTiledFn encode = nullptr;
    // Tensor maps depend only on (base pointer, extent) of q / pool / arena: a model calls msa_forward once per
    // layer with the same few pointer sets step after step, so the 23 encoded maps are kept per pointer set.
    struct MapKey {
        const void *q, *pool_k, *pool_v, *contig_k, *contig_v;
        int64_t total_q, num_blocks, contig_rows;
        bool pool_fp8;
        bool operator==(const MapKey &o) const
        {
            return q == o.q && pool_k == o.pool_k && pool_v == o.pool_v && contig_k == o.contig_k && contig_v == o.contig_v &&
                   total_q == o.total_q && num_blocks == o.num_blocks && contig_rows == o.contig_rows && pool_fp8 == o.pool_fp8;
        }
    };
    struct MapEntry { MapKey key; FwdParams maps; uint64_t stamp; };
    std::vector<MapEntry> map_cache;   // at most kMapCacheEntries, least recently used replaced
    uint64_t map_stamp = 0;
    int last_launches = 0;
    // optional per-launch timing (msa_set_timing): 3 events per recorded step
    bool timing = false;
    std::vector<cudaEvent_t> ev;
    int ev_steps = 0;
    // staging for msa_forward_host / msa_forward_host_async: two slots, so that the upload of one call overlaps the kernels and the
    // read-back of the one before it; copies run on two streams of the handle's own, chained to the caller's stream by events
    struct HostSlot {
        DevBuf s_q, s_o, s_lse, s_ck, s_cv, s_bt, s_ws;
        cudaEvent_t in_done = nullptr, k_done = nullptr, out_done = nullptr;
        bool busy = false;
    };
    HostSlot hs[2];
    cudaStream_t st_in = nullptr, st_out = nullptr;
};

struct msa_plan_s {
    msa_handle h = nullptr;
    int device = -1;                       // the handle's ordinal, kept here: a plan may be destroyed after its handle
    HostPlan hp;
    void *d_buf = nullptr;
    const VBlock *d_vblocks = nullptr;
    const WorkUnit *d_units = nullptr;
    const int32_t *d_cta_begin = nullptr;
    const MergeItem *d_merge = nullptr;
    const TileInfo *d_tile_info = nullptr;
    const int32_t *d_vb_dst = nullptr;     // write-back plans only
    const int32_t *d_tile_writer = nullptr;
    // fp8 pool, plans with pair-mode units: the cached blocks are dequantised once into the workspace (msa_dequant.cu)
    bool deq = false;
    bool any_pair = false;                 // the plan has pair-mode units (which shared-memory layout the fp8 variant needs)
    std::vector<int32_t> deq_src;          // distinct block-table indices the plan refers to; block j of the copy <- deq_src[j]
    std::vector<VBlock> vblocks_deq;       // the plan's virtual blocks with src = index into the copy
    const int32_t *d_deq_src = nullptr;
    const VBlock *d_vblocks_deq = nullptr;
    size_t ws_partials = 0, ws_pool = 0, ws_ident = 0;     // workspace layout in bytes: [partials | copy of K | copy of V | identity table]
    // fp8 pool, write-back plans: the jobs as an append plan of the plan's own -- msa_forward_writeback runs the quantising
    // msa_kv_append kernel behind the forward kernel (the fused store moves bf16 tiles as they are and cannot quantise)
    struct msa_append_plan_s *wb_append = nullptr;
};

struct msa_append_plan_s {
    msa_handle h = nullptr;
    int device = -1;               // as in msa_plan_s
    std::vector<AppendUnit> units;
    AppendUnit *d_units = nullptr;
    int64_t max_row = -1;          // extents the jobs need at msa_kv_append
    int64_t max_bt = -1;
};

extern "C" {

const char *msa_version(void) { return "msa-b200 0.1 (sm_100a)"; }

const char *msa_last_cuda_error(void) { return g_cuda_err.c_str(); }

const char *msa_strerror(int status)
{
    switch (status) {
    case MSA_OK: return "ok";
    case MSA_ERR_INVALID_ARG: return "invalid argument";
    case MSA_ERR_UNSUPPORTED: return "unsupported configuration";
    case MSA_ERR_OVERLAP: return "segments (or q rows) overlap";
    case MSA_ERR_UNSORTED: return "segments not in ascending abs_start";
    case MSA_ERR_OUT_OF_RANGE: return "descriptor out of range";
    case MSA_ERR_MISALIGNED: return "pointer not 16-byte aligned";
    case MSA_ERR_WORKSPACE: return "workspace missing or too small";
    case MSA_ERR_CUDA: return "CUDA error";
    case MSA_ERR_NO_DEVICE: return "no sm_100 CUDA device (there is no CPU fallback)";
    case MSA_ERR_STATIC_WS:
        return "msa_forward_static_ws: the plan needs more scratch than the library's built-in array holds "
               "(MSA_STATIC_WS_BYTES = 32 MiB); pass a workspace of your own to msa_forward";
    default: return "unknown status";
    }
}

int msa_create(const msa_config *cfg, msa_handle *out)
{
    if (!cfg || !out) return MSA_ERR_INVALID_ARG;
    *out = nullptr;
    if (cfg->num_q_heads < 1 || cfg->num_kv_heads < 1) return MSA_ERR_INVALID_ARG;
    if (cfg->head_dim != 64 && cfg->head_dim != 128) return MSA_ERR_UNSUPPORTED;
    if (cfg->block_size != MSA_BLOCK_SIZE) return MSA_ERR_UNSUPPORTED;
    if (cfg->num_q_heads % cfg->num_kv_heads != 0) return MSA_ERR_UNSUPPORTED;
    const int G = cfg->num_q_heads / cfg->num_kv_heads;
    if (G > MSA_MAX_GROUP) return MSA_ERR_UNSUPPORTED;
    if (cfg->pool_format != MSA_POOL_BF16 && cfg->pool_format != MSA_POOL_FP8_E4M3) return MSA_ERR_INVALID_ARG;
    const bool kv8 = cfg->pool_format == MSA_POOL_FP8_E4M3;
    std::vector<float> kv_scale;
    std::vector<uint32_t> kv8_mul;
    std::vector<float> kv8_inv;
    if (kv8) {
        // power-of-two scales only: code * 2^k is exactly a bf16, so the on-chip conversion loses nothing
        for (int which = 0; which < 2; ++which)
            for (int kv = 0; kv < cfg->num_kv_heads; ++kv) {
                const float *src = which ? cfg->v_scale : cfg->k_scale;
                const float sc = src ? src[kv] : 1.f;
                int e = 0;
                if (!(sc > 0.f) || !isfinite(sc)) return MSA_ERR_INVALID_ARG;
                if (frexpf(sc, &e) != 0.5f || e - 1 < -14 || e - 1 > 7) return MSA_ERR_UNSUPPORTED;
                const uint32_t b = static_cast<uint32_t>(15 + (e - 1)) << 10;            // f16 bits of 2^k (normal for k >= -14)
                kv_scale.push_back(sc);
                kv8_mul.push_back(b);
                kv8_inv.push_back(1.f / sc);
            }
    }

    msa_handle h = new (std::nothrow) msa_handle_s();
    if (!h) return MSA_ERR_INVALID_ARG;
    h->cfg = *cfg;
    h->cfg.q_to_kv_head = nullptr;
    h->cfg.k_scale = h->cfg.v_scale = nullptr;
    h->kv8 = kv8;
    h->kv_scale = kv_scale;
    h->G = G;
    h->R = (kTileM / G) & ~7;
    // head map -> q heads of each kv head, in ascending q-head order
    h->kv_to_q.assign(static_cast<size_t>(cfg->num_kv_heads) * G, -1);
    std::vector<int> fill(cfg->num_kv_heads, 0);
    for (int q = 0; q < cfg->num_q_heads; ++q) {
        const int kv = cfg->q_to_kv_head ? cfg->q_to_kv_head[q] : q / G;
        if (kv < 0 || kv >= cfg->num_kv_heads || fill[kv] >= G) {
            delete h;
            return MSA_ERR_UNSUPPORTED;
        }
        h->kv_to_q[static_cast<size_t>(kv) * G + fill[kv]++] = q;
    }
    h->token_major = true;
    for (int kv = 0; kv < cfg->num_kv_heads; ++kv)
        for (int g = 1; g < G; ++g)
            if (h->kv_to_q[static_cast<size_t>(kv) * G + g] != h->kv_to_q[static_cast<size_t>(kv) * G] + g) h->token_major = false;
    if (cfg->device < 0) {
        // planning-only handle: descriptor validation and scheduling on the host; every
        // call that would touch the GPU reports MSA_ERR_NO_DEVICE.
        h->planning_only = true;
        h->num_sms = 148;
        *out = h;
        return MSA_OK;
    }
    int n_dev = 0;
    if (cudaGetDeviceCount(&n_dev) != cudaSuccess || cfg->device >= n_dev) {
        cudaGetLastError();
        delete h;
        return MSA_ERR_NO_DEVICE;
    }
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, cfg->device) != cudaSuccess || prop.major != 10) {
        cudaGetLastError();
        delete h;
        return MSA_ERR_NO_DEVICE;
    }
    h->num_sms = prop.multiProcessorCount;
    DeviceGuard guard(cfg->device);
    cudaError_t e = guard.err;
    if (e == cudaSuccess) e = configure_fwd(cfg->head_dim, kv8);     // per device: a second handle on another GPU sets its own
    if (e == cudaSuccess) e = configure_append();
    if (e == cudaSuccess) e = cudaMalloc(&h->d_kv_to_q, h->kv_to_q.size() * sizeof(int32_t));
    if (e == cudaSuccess)
        e = cudaMemcpy(h->d_kv_to_q, h->kv_to_q.data(), h->kv_to_q.size() * sizeof(int32_t), cudaMemcpyHostToDevice);
    if (kv8) {
        if (e == cudaSuccess) e = cudaMalloc(&h->d_kv8_mul, kv8_mul.size() * sizeof(uint32_t));
        if (e == cudaSuccess) e = cudaMemcpy(h->d_kv8_mul, kv8_mul.data(), kv8_mul.size() * sizeof(uint32_t), cudaMemcpyHostToDevice);
        if (e == cudaSuccess) e = cudaMalloc(&h->d_kv8_inv, kv8_inv.size() * sizeof(float));
        if (e == cudaSuccess) e = cudaMemcpy(h->d_kv8_inv, kv8_inv.data(), kv8_inv.size() * sizeof(float), cudaMemcpyHostToDevice);
    }
    void *fn = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (e == cudaSuccess) e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres);
    if (e != cudaSuccess || !fn) {
        if (h->d_kv_to_q) cudaFree(h->d_kv_to_q);
        if (h->d_kv8_mul) cudaFree(h->d_kv8_mul);
        if (h->d_kv8_inv) cudaFree(h->d_kv8_inv);
        delete h;
        return e != cudaSuccess ? cuda_fail(e, "msa_create") : MSA_ERR_NO_DEVICE;
    }
    h->encode = reinterpret_cast<EncodeTiledFn>(fn);
    h->map_cache.reserve(kMapCacheEntries);      // msa_forward appends to it: no heap traffic on the hot path
    *out = h;
    return MSA_OK;
}

void msa_destroy(msa_handle h)
{
    if (!h) return;
    if (!h->planning_only) {
        DeviceGuard guard(h->cfg.device);
        if (h->d_kv_to_q) cudaFree(h->d_kv_to_q);
        if (h->d_kv8_mul) cudaFree(h->d_kv8_mul);
        if (h->d_kv8_inv) cudaFree(h->d_kv8_inv);
        for (cudaEvent_t e : h->ev) cudaEventDestroy(e);
        for (auto &sl : h->hs) {
            if (sl.busy && sl.out_done) cudaEventSynchronize(sl.out_done);
            sl.s_q.release(); sl.s_o.release(); sl.s_lse.release(); sl.s_ck.release();
            sl.s_cv.release(); sl.s_bt.release(); sl.s_ws.release();
            if (sl.in_done) cudaEventDestroy(sl.in_done);
            if (sl.k_done) cudaEventDestroy(sl.k_done);
            if (sl.out_done) cudaEventDestroy(sl.out_done);
        }
        if (h->st_in) cudaStreamDestroy(h->st_in);
        if (h->st_out) cudaStreamDestroy(h->st_out);
    }
    delete h;
}

}  // extern "C"

namespace {
int plan_create(msa_handle h, const msa_request *requests, int32_t n_req, const msa_segment *segments, int32_t n_seg,
                const msa_append *jobs, int32_t n_jobs, msa_plan *out);
}

extern "C" {

int msa_plan_create(msa_handle h, const msa_request *requests, int32_t n_req, const msa_segment *segments,
                    int32_t n_seg, msa_plan *out)
{
    return plan_create(h, requests, n_req, segments, n_seg, nullptr, 0, out);
}

int msa_plan_create_writeback(msa_handle h, const msa_request *requests, int32_t n_req, const msa_segment *segments,
                              int32_t n_seg, const msa_append *jobs, int32_t n_jobs, msa_plan *out)
{
    if (n_jobs < 0 || (n_jobs > 0 && !jobs)) return MSA_ERR_INVALID_ARG;
    if (h && h->kv8 && n_jobs > 0) {
        // fp8 pool: the same call, two launches (forward kernel, then the quantising append kernel on the same stream)
        if (!out) return MSA_ERR_INVALID_ARG;
        msa_append_plan ap = nullptr;
        int rc = msa_append_plan_create(h, jobs, n_jobs, &ap);
        if (rc != MSA_OK) return rc;
        rc = plan_create(h, requests, n_req, segments, n_seg, nullptr, 0, out);
        if (rc != MSA_OK) {
            msa_append_plan_destroy(ap);
            return rc;
        }
        (*out)->wb_append = ap;
        return MSA_OK;
    }
    return plan_create(h, requests, n_req, segments, n_seg, jobs, n_jobs, out);
}

}  // extern "C"

namespace {

int plan_create(msa_handle h, const msa_request *requests, int32_t n_req, const msa_segment *segments, int32_t n_seg,
                const msa_append *jobs, int32_t n_jobs, msa_plan *out)
{
    if (!h || !out) return MSA_ERR_INVALID_ARG;
    *out = nullptr;
    PlannerConfig pc;
    pc.Hq = h->cfg.num_q_heads;
    pc.Hkv = h->cfg.num_kv_heads;
    pc.D = h->cfg.head_dim;
    pc.G = h->G;
    pc.R = h->R;
    pc.tiles_per_group = kTilesPerGroup;
    pc.num_ctas = h->num_sms;
    msa_plan p = new (std::nothrow) msa_plan_s();
    if (!p) return MSA_ERR_INVALID_ARG;
    p->h = h;
    p->device = h->cfg.device;
    int rc = build_plan(pc, requests, n_req, segments, n_seg, &p->hp, jobs, n_jobs);
    if (rc != MSA_OK) {
        delete p;
        return rc;
    }
    {
        const HostPlan &hp = p->hp;
        p->ws_partials = static_cast<size_t>(hp.workspace_floats) * sizeof(float);
        bool any_pair = false;
        for (const WorkUnit &wu : hp.units) any_pair = any_pair || (wu.mode == kModePair && wu.tile_end > wu.tile_begin);
        p->any_pair = any_pair;
        if (h->kv8 && any_pair && hp.uses_paged) {
            // Dequantising pre-pass (msa_dequant.cu): in a prefill launch a cached tile is loaded by every q-tile group of its
            // (run, KV head), and converting it in the forward kernel repeats the conversion as often.  It pays when the cached
            // blocks are loaded kDeqMinReuse times or more on average: the pre-pass moves 3 bytes per element once and the
            // forward kernel then reads 2 instead of 1 per load.  Compact, sorted list of the block-table entries referred to.
            for (const VBlock &vb : hp.vblocks)
                if (vb.paged && vb.nvalid > 0) p->deq_src.push_back(vb.src);
            std::sort(p->deq_src.begin(), p->deq_src.end());
            p->deq_src.erase(std::unique(p->deq_src.begin(), p->deq_src.end()), p->deq_src.end());
            int64_t loads = 0;                 // (cached 16-token block, KV head) pairs loaded by the launch, over all units
            for (const WorkUnit &wu : hp.units)
                for (int t = wu.tile_begin; t < wu.tile_end; ++t)
                    for (int b = 0; b < kVbPerTile; ++b) {
                        const int i = t * kVbPerTile + b;
                        if (i < wu.vb_count && hp.vblocks[wu.vb_begin + i].paged && hp.vblocks[wu.vb_begin + i].nvalid > 0) ++loads;
                    }
            constexpr double kDeqMinReuse = 2.0;
            p->deq = !p->deq_src.empty() &&
                     static_cast<double>(loads) >= kDeqMinReuse * static_cast<double>(p->deq_src.size()) * h->cfg.num_kv_heads;
            if (!p->deq) p->deq_src.clear();
        }
        if (p->deq) {
            p->vblocks_deq = hp.vblocks;
            for (VBlock &vb : p->vblocks_deq)
                if (vb.paged && vb.nvalid > 0)
                    vb.src = static_cast<int32_t>(std::lower_bound(p->deq_src.begin(), p->deq_src.end(), vb.src) - p->deq_src.begin());
            auto al1k = [](size_t x) { return (x + 1023) & ~static_cast<size_t>(1023); };
            p->ws_partials = al1k(p->ws_partials);
            p->ws_pool = al1k(p->deq_src.size() * static_cast<size_t>(MSA_BLOCK_SIZE) * h->cfg.num_kv_heads * h->cfg.head_dim * 2);
            p->ws_ident = al1k(p->deq_src.size() * sizeof(int32_t));
        }
    }
    if (!h->planning_only) {
        const HostPlan &hp = p->hp;
        auto al = [](size_t x) { return (x + 255) & ~static_cast<size_t>(255); };
        const size_t b_vb = al(hp.vblocks.size() * sizeof(VBlock));
        const size_t b_un = al(hp.units.size() * sizeof(WorkUnit));
        const size_t b_cb = al(hp.cta_unit_begin.size() * sizeof(int32_t));
        const size_t b_mg = al(hp.merge_items.size() * sizeof(MergeItem));
        const size_t b_ti = al(hp.tile_info.size() * sizeof(TileInfo));
        const size_t b_wb = al(hp.vb_dst.size() * sizeof(int32_t));
        const size_t b_tw = al(hp.tile_writer.size() * sizeof(int32_t));
        const size_t b_ds = al(p->deq_src.size() * sizeof(int32_t));
        const size_t b_vd = al(p->vblocks_deq.size() * sizeof(VBlock));
        const size_t total = b_vb + b_un + b_cb + b_mg + b_ti + b_wb + b_tw + b_ds + b_vd + 256;
        DeviceGuard guard(h->cfg.device);
        cudaError_t e = guard.err;
        if (e == cudaSuccess) e = cudaMalloc(&p->d_buf, total);
        if (e != cudaSuccess) {
            delete p;
            return cuda_fail(e, "msa_plan_create: cudaMalloc");
        }
        char *base = static_cast<char *>(p->d_buf);
        p->d_vblocks = reinterpret_cast<const VBlock *>(base);
        p->d_units = reinterpret_cast<const WorkUnit *>(base + b_vb);
        p->d_cta_begin = reinterpret_cast<const int32_t *>(base + b_vb + b_un);
        p->d_merge = reinterpret_cast<const MergeItem *>(base + b_vb + b_un + b_cb);
        p->d_tile_info = reinterpret_cast<const TileInfo *>(base + b_vb + b_un + b_cb + b_mg);
        if (hp.has_writeback) {
            p->d_vb_dst = reinterpret_cast<const int32_t *>(base + b_vb + b_un + b_cb + b_mg + b_ti);
            p->d_tile_writer = reinterpret_cast<const int32_t *>(base + b_vb + b_un + b_cb + b_mg + b_ti + b_wb);
        }
        if (e == cudaSuccess && !hp.vblocks.empty())
            e = cudaMemcpy(base, hp.vblocks.data(), hp.vblocks.size() * sizeof(VBlock), cudaMemcpyHostToDevice);
        if (e == cudaSuccess && !hp.units.empty())
            e = cudaMemcpy(base + b_vb, hp.units.data(), hp.units.size() * sizeof(WorkUnit), cudaMemcpyHostToDevice);
        if (e == cudaSuccess && !hp.cta_unit_begin.empty())
            e = cudaMemcpy(base + b_vb + b_un, hp.cta_unit_begin.data(), hp.cta_unit_begin.size() * sizeof(int32_t),
                           cudaMemcpyHostToDevice);
        if (e == cudaSuccess && !hp.merge_items.empty())
            e = cudaMemcpy(base + b_vb + b_un + b_cb, hp.merge_items.data(), hp.merge_items.size() * sizeof(MergeItem),
                           cudaMemcpyHostToDevice);
        if (e == cudaSuccess && !hp.tile_info.empty())
            e = cudaMemcpy(base + b_vb + b_un + b_cb + b_mg, hp.tile_info.data(), hp.tile_info.size() * sizeof(TileInfo),
                           cudaMemcpyHostToDevice);
        if (e == cudaSuccess && !hp.vb_dst.empty())
            e = cudaMemcpy(base + b_vb + b_un + b_cb + b_mg + b_ti, hp.vb_dst.data(), hp.vb_dst.size() * sizeof(int32_t),
                           cudaMemcpyHostToDevice);
        if (e == cudaSuccess && !hp.tile_writer.empty())
            e = cudaMemcpy(base + b_vb + b_un + b_cb + b_mg + b_ti + b_wb, hp.tile_writer.data(), hp.tile_writer.size() * sizeof(int32_t),
                           cudaMemcpyHostToDevice);
        if (p->deq) {
            char *ds = base + b_vb + b_un + b_cb + b_mg + b_ti + b_wb + b_tw;
            p->d_deq_src = reinterpret_cast<const int32_t *>(ds);
            p->d_vblocks_deq = reinterpret_cast<const VBlock *>(ds + b_ds);
            if (e == cudaSuccess && !p->deq_src.empty())
                e = cudaMemcpy(ds, p->deq_src.data(), p->deq_src.size() * sizeof(int32_t), cudaMemcpyHostToDevice);
            if (e == cudaSuccess && !p->vblocks_deq.empty())
                e = cudaMemcpy(ds + b_ds, p->vblocks_deq.data(), p->vblocks_deq.size() * sizeof(VBlock), cudaMemcpyHostToDevice);
        }
        if (e != cudaSuccess) {
            cudaFree(p->d_buf);
            delete p;
            return cuda_fail(e, "msa_plan_create: upload");
        }
    }
    *out = p;
    return MSA_OK;
}

}  // namespace

extern "C" {

void msa_plan_destroy(msa_plan p)
{
    if (!p) return;
    if (p->wb_append) msa_append_plan_destroy(p->wb_append);
    if (p->d_buf) {
        DeviceGuard guard(p->device);
        cudaFree(p->d_buf);
    }
    delete p;
}

int msa_plan_get_info(msa_plan p, msa_plan_info *info)
{
    if (!p || !info) return MSA_ERR_INVALID_ARG;
    *info = p->hp.info;
    return MSA_OK;
}

int msa_workspace_bytes(msa_plan p, size_t *bytes)
{
    if (!p || !bytes) return MSA_ERR_INVALID_ARG;
    *bytes = p->ws_partials + 2 * p->ws_pool + p->ws_ident;
    return MSA_OK;
}

/* Introspection for tests: copies the host-side plan arrays out.
 * which: 0 = virtual blocks (int32 x4 each), 1 = work units (int32 x12 each),
 *        2 = cta_unit_begin (int32), 3 = merge items (int32 x4 + int64 x2 each),
 *        4 = per-tile mask summaries (int32 x2 each), 5 / 6 = write-back plans: destination block-table index per
 *        virtual block, q_row0 of the storing work item per context KV tile (int32 each); 7 = fp8 pool: the block-table
 *        indices the dequantising pre-pass converts (int32 each; empty when the forward kernel converts the codes itself).
 * Call with buf == NULL to get the byte size. */
int msa_plan_export(msa_plan p, int which, void *buf, size_t *bytes)
{
    if (!p || !bytes) return MSA_ERR_INVALID_ARG;
    const void *src = nullptr;
    size_t n = 0;
    switch (which) {
    case 0: src = p->hp.vblocks.data(); n = p->hp.vblocks.size() * sizeof(VBlock); break;
    case 1: src = p->hp.units.data(); n = p->hp.units.size() * sizeof(WorkUnit); break;
    case 2: src = p->hp.cta_unit_begin.data(); n = p->hp.cta_unit_begin.size() * sizeof(int32_t); break;
    case 3: src = p->hp.merge_items.data(); n = p->hp.merge_items.size() * sizeof(MergeItem); break;
    case 4: src = p->hp.tile_info.data(); n = p->hp.tile_info.size() * sizeof(TileInfo); break;
    case 5: src = p->hp.vb_dst.data(); n = p->hp.vb_dst.size() * sizeof(int32_t); break;
    case 6: src = p->hp.tile_writer.data(); n = p->hp.tile_writer.size() * sizeof(int32_t); break;
    case 7: src = p->deq_src.data(); n = p->deq_src.size() * sizeof(int32_t); break;
    default: return MSA_ERR_INVALID_ARG;
    }
    if (buf) {
        if (*bytes < n) return MSA_ERR_INVALID_ARG;
        if (n) memcpy(buf, src, n);
    }
    *bytes = n;
    return MSA_OK;
}

}  // extern "C"

namespace {

int encode_2d(msa_handle h, CUtensorMap *tm, const void *base, uint64_t inner_elems, uint64_t rows, uint32_t box_rows)
{
    cuuint64_t gdim[2] = {inner_elems, rows > 0 ? rows : 1};
    cuuint64_t gstride[1] = {inner_elems * 2};
    cuuint32_t box[2] = {64, box_rows};
    cuuint32_t estr[2] = {1, 1};
    CUresult r = h->encode(tm, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<void *>(base), gdim, gstride, box, estr,
                           CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                           CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) {
        char msg[96];
        snprintf(msg, sizeof msg, "cuTensorMapEncodeTiled failed: CUresult %d", static_cast<int>(r));
        g_cuda_err = msg;
        return MSA_ERR_CUDA;
    }
    return MSA_OK;
}

// fp8 pool: bytes [rows][inner], box = head_dim bytes x box_rows, no swizzle (the converter warps read the staging slot
// with plain 16-byte shared loads)
int encode_2d_u8(msa_handle h, CUtensorMap *tm, const void *base, uint64_t inner_bytes, uint64_t rows, uint32_t box_inner,
                 uint32_t box_rows)
{
    cuuint64_t gdim[2] = {inner_bytes, rows > 0 ? rows : 1};
    cuuint64_t gstride[1] = {inner_bytes};
    cuuint32_t box[2] = {box_inner, box_rows};
    cuuint32_t estr[2] = {1, 1};
    CUresult r = h->encode(tm, CU_TENSOR_MAP_DATA_TYPE_UINT8, 2, const_cast<void *>(base), gdim, gstride, box, estr,
                           CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                           CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) {
        char msg[96];
        snprintf(msg, sizeof msg, "cuTensorMapEncodeTiled (u8) failed: CUresult %d", static_cast<int>(r));
        g_cuda_err = msg;
        return MSA_ERR_CUDA;
    }
    return MSA_OK;
}

bool aligned16(const void *p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

// The 23 tensor maps of one (q, pool, arena) pointer set, encoded once and kept in the handle.
int cached_tensor_maps(msa_handle h, const HostPlan &hp_in, bool writeback, bool pool_fp8, const void *q, int64_t total_q,
                       const void *pool_k, const void *pool_v, int64_t num_blocks, const void *contig_k, const void *contig_v,
                       int64_t contig_rows, FwdParams *out)
{
    const int Hq = h->cfg.num_q_heads, Hkv = h->cfg.num_kv_heads, D = h->cfg.head_dim;
    struct { bool uses_paged, uses_contig; } hp{hp_in.uses_paged || writeback, hp_in.uses_contig};   // write-back stores through the pool maps
    // a plan that uses no paged (or no contiguous) segment never dereferences those maps: they are encoded over q
    msa_handle_s::MapKey key{q, hp.uses_paged ? pool_k : nullptr, hp.uses_paged ? pool_v : nullptr,
                             hp.uses_contig ? contig_k : nullptr, hp.uses_contig ? contig_v : nullptr,
                             total_q, hp.uses_paged ? num_blocks : 0, hp.uses_contig ? contig_rows : 0, pool_fp8};
    ++h->map_stamp;
    for (auto &e : h->map_cache)
        if (e.key == key) {
            e.stamp = h->map_stamp;
            *out = e.maps;
            return MSA_OK;
        }
    FwdParams fp;
    memset(&fp, 0, sizeof fp);
    int rc = encode_2d(h, &fp.tm_q, q, static_cast<uint64_t>(Hq) * D, static_cast<uint64_t>(total_q), h->R);
    if (rc != MSA_OK) return rc;
    {   // q as [total_q][Hq][D]: box = 64 elements x G heads x R tokens, rows land token-major
        cuuint64_t gdim[3] = {static_cast<cuuint64_t>(D), static_cast<cuuint64_t>(Hq), static_cast<cuuint64_t>(total_q > 0 ? total_q : 1)};
        cuuint64_t gstride[2] = {static_cast<cuuint64_t>(D) * 2, static_cast<cuuint64_t>(Hq) * D * 2};
        cuuint32_t box[3] = {64, static_cast<cuuint32_t>(h->G), static_cast<cuuint32_t>(h->R)};
        cuuint32_t estr[3] = {1, 1, 1};
        CUresult r = h->encode(&fp.tm_q3, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 3, const_cast<void *>(q), gdim, gstride, box, estr,
                               CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                               CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        if (r != CUDA_SUCCESS) {
            char msg[96];
            snprintf(msg, sizeof msg, "cuTensorMapEncodeTiled (q, 3-D) failed: CUresult %d", static_cast<int>(r));
            g_cuda_err = msg;
            return MSA_ERR_CUDA;
        }
    }
    const void *pk = hp.uses_paged ? pool_k : q;
    const void *pv = hp.uses_paged ? pool_v : q;
    const uint64_t prow = hp.uses_paged ? static_cast<uint64_t>(num_blocks) * MSA_BLOCK_SIZE : static_cast<uint64_t>(total_q);
    const uint64_t pin = hp.uses_paged ? static_cast<uint64_t>(Hkv) * D : static_cast<uint64_t>(Hq) * D;
    for (int i = 0; i < 5; ++i) {
        if (pool_fp8 && hp.uses_paged) {
            if ((rc = encode_2d_u8(h, &fp.tm_pool_k[i], pk, pin, prow, D, MSA_BLOCK_SIZE >> i)) != MSA_OK) return rc;
            if ((rc = encode_2d_u8(h, &fp.tm_pool_v[i], pv, pin, prow, D, MSA_BLOCK_SIZE >> i)) != MSA_OK) return rc;
            continue;
        }
        if ((rc = encode_2d(h, &fp.tm_pool_k[i], pk, pin, prow, MSA_BLOCK_SIZE >> i)) != MSA_OK) return rc;
        if ((rc = encode_2d(h, &fp.tm_pool_v[i], pv, pin, prow, MSA_BLOCK_SIZE >> i)) != MSA_OK) return rc;
    }
    const void *ck = hp.uses_contig ? contig_k : q;
    const void *cv = hp.uses_contig ? contig_v : q;
    const uint64_t crow = hp.uses_contig ? static_cast<uint64_t>(contig_rows) : static_cast<uint64_t>(total_q);
    const uint64_t cin = hp.uses_contig ? static_cast<uint64_t>(Hkv) * D : static_cast<uint64_t>(Hq) * D;
    for (int i = 0; i < 5; ++i) {
        if ((rc = encode_2d(h, &fp.tm_ctg_k[i], ck, cin, crow, MSA_BLOCK_SIZE >> i)) != MSA_OK) return rc;
        if ((rc = encode_2d(h, &fp.tm_ctg_v[i], cv, cin, crow, MSA_BLOCK_SIZE >> i)) != MSA_OK) return rc;
    }
    if ((rc = encode_2d(h, &fp.tm_ctg_k128, ck, cin, crow, kTileN)) != MSA_OK) return rc;
    if ((rc = encode_2d(h, &fp.tm_ctg_v128, cv, cin, crow, kTileN)) != MSA_OK) return rc;
    if (h->map_cache.size() < kMapCacheEntries) {
        h->map_cache.push_back({key, fp, h->map_stamp});
    } else {
        auto victim = std::min_element(h->map_cache.begin(), h->map_cache.end(),
                                       [](const msa_handle_s::MapEntry &a, const msa_handle_s::MapEntry &b) { return a.stamp < b.stamp; });
        *victim = {key, fp, h->map_stamp};
    }
    *out = fp;
    return MSA_OK;
}

}  // namespace

namespace {

int forward_impl(msa_handle h, msa_plan p, const void *q, int64_t total_q, const void *pool_k, const void *pool_v,
                 int64_t num_blocks, const int32_t *block_table, int64_t block_table_len, const void *contig_k,
                 const void *contig_v, int64_t contig_rows, float softmax_scale, void *o, float *lse, void *workspace,
                 size_t workspace_bytes, void *cuda_stream, bool writeback)
{
    if (!h || !p || p->h != h) return MSA_ERR_INVALID_ARG;
    if (h->planning_only) return MSA_ERR_NO_DEVICE;
    h->last_launches = 0;
    const HostPlan &hp = p->hp;
    if (writeback && h->kv8) {
        // fp8 pool: forward (no fused store), then the plan's own append plan through the quantising kernel, same stream
        if (!p->wb_append) return MSA_ERR_INVALID_ARG;
        if (!pool_k || !pool_v || !block_table || num_blocks < 1) return MSA_ERR_INVALID_ARG;
        if (p->wb_append->max_bt >= block_table_len || p->wb_append->max_row >= contig_rows) return MSA_ERR_OUT_OF_RANGE;
        int rc = forward_impl(h, p, q, total_q, pool_k, pool_v, num_blocks, block_table, block_table_len, contig_k, contig_v,
                              contig_rows, softmax_scale, o, lse, workspace, workspace_bytes, cuda_stream, false);
        if (rc != MSA_OK) return rc;
        const int fwd_launches = h->last_launches;
        rc = msa_kv_append(h, p->wb_append, contig_k, contig_v, contig_rows, const_cast<void *>(pool_k), const_cast<void *>(pool_v),
                           num_blocks, block_table, block_table_len, cuda_stream);
        if (rc != MSA_OK) return rc;
        h->last_launches += fwd_launches;
        return MSA_OK;
    }
    if (writeback) {
        if (!hp.has_writeback) return MSA_ERR_INVALID_ARG;          // the plan must come from msa_plan_create_writeback
        if (!pool_k || !pool_v || !block_table || num_blocks < 1 || num_blocks * MSA_BLOCK_SIZE > 0x7fffffffLL) return MSA_ERR_INVALID_ARG;
        if (hp.wb_max_bt >= block_table_len) return MSA_ERR_OUT_OF_RANGE;
    }
    if (!(softmax_scale > 0.f) || !isfinite(softmax_scale)) return MSA_ERR_INVALID_ARG;
    if (total_q < 0 || num_blocks < 0 || block_table_len < 0 || contig_rows < 0) return MSA_ERR_INVALID_ARG;
    if (hp.info.num_units == 0) return MSA_OK;
    if (!q || !o || !lse) return MSA_ERR_INVALID_ARG;
    if (hp.uses_paged && (!pool_k || !pool_v || !block_table)) return MSA_ERR_INVALID_ARG;
    if (hp.uses_contig && (!contig_k || !contig_v)) return MSA_ERR_INVALID_ARG;
    if (hp.info.max_q_row >= total_q) return MSA_ERR_OUT_OF_RANGE;
    if (hp.uses_paged && hp.info.max_block_table_index >= block_table_len) return MSA_ERR_OUT_OF_RANGE;
    if (hp.uses_contig && hp.info.max_contig_row >= contig_rows) return MSA_ERR_OUT_OF_RANGE;
    if (hp.uses_paged && (num_blocks < 1 || num_blocks * MSA_BLOCK_SIZE > 0x7fffffffLL)) return MSA_ERR_OUT_OF_RANGE;
    if (!aligned16(q) || !aligned16(o) || !aligned16(pool_k) || !aligned16(pool_v) || !aligned16(contig_k) ||
        !aligned16(contig_v) || (reinterpret_cast<uintptr_t>(lse) & 3u) || (reinterpret_cast<uintptr_t>(block_table) & 3u))
        return MSA_ERR_MISALIGNED;
    const size_t need = p->ws_partials + 2 * p->ws_pool + p->ws_ident;
    if (need > 0) {
        if (!workspace || workspace_bytes < need) return MSA_ERR_WORKSPACE;
        if (!aligned16(workspace)) return MSA_ERR_MISALIGNED;
    }

    const int Hq = h->cfg.num_q_heads, Hkv = h->cfg.num_kv_heads, D = h->cfg.head_dim;
    DeviceGuard guard(h->cfg.device);      // the caller's current device may be another one
    if (guard.err != cudaSuccess) return cuda_fail(guard.err, "msa_forward: cudaSetDevice");
    // fp8 pool and prefill units: the cached blocks are dequantised once into the workspace, the bf16 kernel runs on that copy
    char *ws = static_cast<char *>(workspace);
    void *copy_k = p->deq ? ws + p->ws_partials : nullptr, *copy_v = p->deq ? ws + p->ws_partials + p->ws_pool : nullptr;
    int32_t *ident = p->deq ? reinterpret_cast<int32_t *>(ws + p->ws_partials + 2 * p->ws_pool) : nullptr;
    const bool pool_fp8 = h->kv8 && !p->deq && hp.uses_paged;     // no cached segment in the plan: nothing to convert, the bf16 kernel
    FwdParams fp;
    int rc = p->deq ? cached_tensor_maps(h, hp, false, false, q, total_q, copy_k, copy_v, static_cast<int64_t>(p->deq_src.size()), contig_k,
                                         contig_v, contig_rows, &fp)
                    : cached_tensor_maps(h, hp, writeback, pool_fp8, q, total_q, pool_k, pool_v, num_blocks, contig_k, contig_v,
                                         contig_rows, &fp);
    if (rc != MSA_OK) return rc;
    fp.vblocks = p->deq ? p->d_vblocks_deq : p->d_vblocks;
    fp.units = p->d_units;
    fp.cta_unit_begin = p->d_cta_begin;
    fp.tile_info = p->d_tile_info;
    fp.block_table = p->deq ? ident : block_table;
    fp.vb_dst = writeback ? p->d_vb_dst : nullptr;
    fp.tile_writer = writeback ? p->d_tile_writer : nullptr;
    fp.kv_to_q = h->d_kv_to_q;
    fp.kv8_mul = h->d_kv8_mul;
    fp.o = o;
    fp.lse = lse;
    fp.workspace = static_cast<float *>(workspace);
    fp.scale_log2 = softmax_scale * 1.4426950408889634f;
    fp.Hq = Hq;
    fp.Hkv = Hkv;
    fp.G = h->G;
    fp.R = h->R;
    fp.token_major = h->token_major ? 1 : 0;
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    const bool rec = h->timing && static_cast<size_t>(h->ev_steps) * 3 + 3 <= h->ev.size();
    cudaEvent_t *ev = rec ? &h->ev[static_cast<size_t>(h->ev_steps) * 3] : nullptr;
    if (rec) MSA_CUDA(cudaEventRecord(ev[0], stream));
    int launches = 0;
    if (p->deq) {
        DequantParams dq;
        dq.src_bt = p->d_deq_src;
        dq.block_table = block_table;
        dq.pool_k = pool_k;
        dq.pool_v = pool_v;
        dq.out_k = copy_k;
        dq.out_v = copy_v;
        dq.ident = ident;
        dq.kv8_mul = h->d_kv8_mul;
        dq.n_blocks = static_cast<int32_t>(p->deq_src.size());
        dq.Hkv = Hkv;
        dq.D = D;
        MSA_CUDA(launch_dequant(dq, h->num_sms, stream));
        ++launches;
    }
    MSA_CUDA(launch_fwd(fp, D, pool_fp8, !p->any_pair, hp.info.num_ctas, stream));
    if (rec) MSA_CUDA(cudaEventRecord(ev[1], stream));
    h->last_launches = ++launches;
    if (!hp.merge_items.empty()) {
        MergeParams mp;
        mp.items = p->d_merge;
        mp.kv_to_q = h->d_kv_to_q;
        mp.workspace = static_cast<const float *>(workspace);
        mp.o = o;
        mp.lse = lse;
        mp.Hq = Hq;
        mp.G = h->G;
        mp.D = D;
        int max_rows = 0;
        for (const MergeItem &mi : hp.merge_items) max_rows = std::max(max_rows, mi.n_tok * h->G);
        MSA_CUDA(launch_merge(mp, static_cast<int>(hp.merge_items.size()), max_rows, stream));
        h->last_launches = ++launches;
    }
    if (rec) {
        MSA_CUDA(cudaEventRecord(ev[2], stream));
        ++h->ev_steps;
    }
    return MSA_OK;
}

}  // namespace

extern "C" {

int msa_forward(msa_handle h, msa_plan p, const void *q, int64_t total_q, const void *pool_k, const void *pool_v,
                int64_t num_blocks, const int32_t *block_table, int64_t block_table_len, const void *contig_k,
                const void *contig_v, int64_t contig_rows, float softmax_scale, void *o, float *lse, void *workspace,
                size_t workspace_bytes, void *cuda_stream)
{
    return forward_impl(h, p, q, total_q, pool_k, pool_v, num_blocks, block_table, block_table_len, contig_k, contig_v, contig_rows,
                        softmax_scale, o, lse, workspace, workspace_bytes, cuda_stream, false);
}

int msa_forward_writeback(msa_handle h, msa_plan p, const void *q, int64_t total_q, void *pool_k, void *pool_v, int64_t num_blocks,
                          const int32_t *block_table, int64_t block_table_len, const void *contig_k, const void *contig_v,
                          int64_t contig_rows, float softmax_scale, void *o, float *lse, void *workspace, size_t workspace_bytes,
                          void *cuda_stream)
{
    return forward_impl(h, p, q, total_q, pool_k, pool_v, num_blocks, block_table, block_table_len, contig_k, contig_v, contig_rows,
                        softmax_scale, o, lse, workspace, workspace_bytes, cuda_stream, true);
}

int msa_forward_host_async(msa_handle h, msa_plan p, const void *q_host, int64_t total_q, const void *pool_k,
                           const void *pool_v, int64_t num_blocks, const int32_t *block_table_host, int64_t block_table_len,
                           const void *contig_k_host, const void *contig_v_host, int64_t contig_rows, float softmax_scale,
                           void *o_host, float *lse_host, void *cuda_stream, int32_t slot)
{
    if (!h || !p || p->h != h || slot < 0 || slot > 1) return MSA_ERR_INVALID_ARG;
    if (h->planning_only) return MSA_ERR_NO_DEVICE;
    if (total_q < 0 || block_table_len < 0 || contig_rows < 0) return MSA_ERR_INVALID_ARG;
    if (total_q > 0 && (!q_host || !o_host || !lse_host)) return MSA_ERR_INVALID_ARG;
    if (block_table_len > 0 && !block_table_host) return MSA_ERR_INVALID_ARG;
    if (contig_rows > 0 && (!contig_k_host || !contig_v_host)) return MSA_ERR_INVALID_ARG;
    const int Hq = h->cfg.num_q_heads, Hkv = h->cfg.num_kv_heads, D = h->cfg.head_dim;
    const size_t b_q = static_cast<size_t>(total_q) * Hq * D * 2;
    const size_t b_lse = static_cast<size_t>(total_q) * Hq * 4;
    const size_t b_c = static_cast<size_t>(contig_rows) * Hkv * D * 2;
    const size_t b_bt = static_cast<size_t>(block_table_len) * 4;
    const size_t b_ws = p->ws_partials + 2 * p->ws_pool + p->ws_ident;
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    DeviceGuard guard(h->cfg.device);
    if (guard.err != cudaSuccess) return cuda_fail(guard.err, "msa_forward_host: cudaSetDevice");
    if (!h->st_in) MSA_CUDA(cudaStreamCreateWithFlags(&h->st_in, cudaStreamNonBlocking));
    if (!h->st_out) MSA_CUDA(cudaStreamCreateWithFlags(&h->st_out, cudaStreamNonBlocking));
    msa_handle_s::HostSlot &sl = h->hs[slot];
    // a staging buffer that is about to be re-allocated takes the tensor maps encoded over it with it
    if (b_q + 16 > sl.s_q.cap || b_c + 16 > sl.s_ck.cap || b_c + 16 > sl.s_cv.cap) {
        const void *gone[3] = {sl.s_q.p, sl.s_ck.p, sl.s_cv.p};
        h->map_cache.erase(std::remove_if(h->map_cache.begin(), h->map_cache.end(),
                                          [&](const msa_handle_s::MapEntry &e) {
                                              for (const void *g : gone)
                                                  if (g && (e.key.q == g || e.key.contig_k == g || e.key.contig_v == g)) return true;
                                              return false;
                                          }),
                           h->map_cache.end());
    }
    if (!sl.in_done) MSA_CUDA(cudaEventCreateWithFlags(&sl.in_done, cudaEventDisableTiming));
    if (!sl.k_done) MSA_CUDA(cudaEventCreateWithFlags(&sl.k_done, cudaEventDisableTiming));
    if (!sl.out_done) MSA_CUDA(cudaEventCreateWithFlags(&sl.out_done, cudaEventDisableTiming));
    // the slot's last call must be over before its staging buffers (and the caller's output buffers) are used again
    if (sl.busy) MSA_CUDA(cudaEventSynchronize(sl.out_done));
    sl.busy = false;
    MSA_CUDA(sl.s_q.reserve(b_q + 16));
    MSA_CUDA(sl.s_o.reserve(b_q + 16));
    MSA_CUDA(sl.s_lse.reserve(b_lse + 16));
    MSA_CUDA(sl.s_ck.reserve(b_c + 16));
    MSA_CUDA(sl.s_cv.reserve(b_c + 16));
    MSA_CUDA(sl.s_bt.reserve(b_bt + 16));
    MSA_CUDA(sl.s_ws.reserve(b_ws + 16));
    if (b_q) MSA_CUDA(cudaMemcpyAsync(sl.s_q.p, q_host, b_q, cudaMemcpyHostToDevice, h->st_in));
    if (b_bt) MSA_CUDA(cudaMemcpyAsync(sl.s_bt.p, block_table_host, b_bt, cudaMemcpyHostToDevice, h->st_in));
    if (b_c) {
        MSA_CUDA(cudaMemcpyAsync(sl.s_ck.p, contig_k_host, b_c, cudaMemcpyHostToDevice, h->st_in));
        MSA_CUDA(cudaMemcpyAsync(sl.s_cv.p, contig_v_host, b_c, cudaMemcpyHostToDevice, h->st_in));
    }
    MSA_CUDA(cudaEventRecord(sl.in_done, h->st_in));
    MSA_CUDA(cudaStreamWaitEvent(stream, sl.in_done, 0));
    int rc = msa_forward(h, p, sl.s_q.p, total_q, pool_k, pool_v, num_blocks, static_cast<const int32_t *>(sl.s_bt.p),
                         block_table_len, sl.s_ck.p, sl.s_cv.p, contig_rows, softmax_scale, sl.s_o.p,
                         static_cast<float *>(sl.s_lse.p), sl.s_ws.p, sl.s_ws.cap, stream);
    if (rc != MSA_OK) return rc;
    MSA_CUDA(cudaEventRecord(sl.k_done, stream));
    MSA_CUDA(cudaStreamWaitEvent(h->st_out, sl.k_done, 0));
    if (b_q) {
        MSA_CUDA(cudaMemcpyAsync(o_host, sl.s_o.p, b_q, cudaMemcpyDeviceToHost, h->st_out));
        MSA_CUDA(cudaMemcpyAsync(lse_host, sl.s_lse.p, b_lse, cudaMemcpyDeviceToHost, h->st_out));
    }
    MSA_CUDA(cudaEventRecord(sl.out_done, h->st_out));
    sl.busy = true;
    return MSA_OK;
}

int msa_forward_host_wait(msa_handle h, int32_t slot)
{
    if (!h || slot < 0 || slot > 1) return MSA_ERR_INVALID_ARG;
    if (h->planning_only) return MSA_ERR_NO_DEVICE;
    msa_handle_s::HostSlot &sl = h->hs[slot];
    if (!sl.busy) return MSA_OK;
    DeviceGuard guard(h->cfg.device);
    if (guard.err != cudaSuccess) return cuda_fail(guard.err, "msa_forward_host_wait: cudaSetDevice");
    MSA_CUDA(cudaEventSynchronize(sl.out_done));
    sl.busy = false;
    return MSA_OK;
}

int msa_forward_host(msa_handle h, msa_plan p, const void *q_host, int64_t total_q, const void *pool_k,
                     const void *pool_v, int64_t num_blocks, const int32_t *block_table_host, int64_t block_table_len,
                     const void *contig_k_host, const void *contig_v_host, int64_t contig_rows, float softmax_scale,
                     void *o_host, float *lse_host, void *cuda_stream)
{
    int rc = msa_forward_host_async(h, p, q_host, total_q, pool_k, pool_v, num_blocks, block_table_host, block_table_len, contig_k_host,
                                    contig_v_host, contig_rows, softmax_scale, o_host, lse_host, cuda_stream, 0);
    if (rc != MSA_OK) return rc;
    return msa_forward_host_wait(h, 0);
}

int msa_append_plan_create(msa_handle h, const msa_append *jobs, int32_t n_jobs, msa_append_plan *out)
{
    if (!h || !out || n_jobs < 0 || (n_jobs > 0 && !jobs)) return MSA_ERR_INVALID_ARG;
    *out = nullptr;
    msa_append_plan ap = new (std::nothrow) msa_append_plan_s();
    if (!ap) return MSA_ERR_INVALID_ARG;
    ap->h = h;
    ap->device = h->cfg.device;
    std::vector<std::pair<int64_t, int64_t>> spans;      // destination block-table ranges, for the overlap check
    for (int32_t j = 0; j < n_jobs; ++j) {
        const msa_append &a = jobs[j];
        if (a.len < 1 || a.row_off < 0 || a.block_off < 0) {
            delete ap;
            return MSA_ERR_INVALID_ARG;
        }
        const int nblk = (a.len + kBlock - 1) / kBlock;
        const int64_t last_bt = static_cast<int64_t>(a.block_off) + nblk - 1;
        if (last_bt > INT32_MAX || a.row_off + a.len - 1 > INT32_MAX) {
            delete ap;
            return MSA_ERR_OUT_OF_RANGE;
        }
        spans.emplace_back(a.block_off, last_bt + 1);
        ap->max_bt = std::max(ap->max_bt, last_bt);
        ap->max_row = std::max(ap->max_row, a.row_off + a.len - 1);
        for (int b = 0; b < nblk; ++b) {
            AppendUnit u;
            u.src_row = a.row_off + static_cast<int64_t>(b) * kBlock;
            u.bt_index = a.block_off + b;
            u.nvalid = std::min(kBlock, a.len - b * kBlock);
            ap->units.push_back(u);
        }
    }
    std::sort(spans.begin(), spans.end());
    for (size_t i = 1; i < spans.size(); ++i)
        if (spans[i].first < spans[i - 1].second) {
            delete ap;
            return MSA_ERR_OVERLAP;
        }
    if (!h->planning_only && !ap->units.empty()) {
        DeviceGuard guard(h->cfg.device);
        cudaError_t e = guard.err;
        if (e == cudaSuccess) e = cudaMalloc(&ap->d_units, ap->units.size() * sizeof(AppendUnit));
        if (e == cudaSuccess)
            e = cudaMemcpy(ap->d_units, ap->units.data(), ap->units.size() * sizeof(AppendUnit), cudaMemcpyHostToDevice);
        if (e != cudaSuccess) {
            if (ap->d_units) cudaFree(ap->d_units);
            delete ap;
            return cuda_fail(e, "msa_append_plan_create: upload");
        }
    }
    *out = ap;
    return MSA_OK;
}

void msa_append_plan_destroy(msa_append_plan ap)
{
    if (!ap) return;
    if (ap->d_units) {
        DeviceGuard guard(ap->device);
        cudaFree(ap->d_units);
    }
    delete ap;
}

int msa_kv_append(msa_handle h, msa_append_plan ap, const void *contig_k, const void *contig_v, int64_t contig_rows,
                  void *pool_k, void *pool_v, int64_t num_blocks, const int32_t *block_table, int64_t block_table_len,
                  void *cuda_stream)
{
    if (!h || !ap || ap->h != h) return MSA_ERR_INVALID_ARG;
    if (h->planning_only) return MSA_ERR_NO_DEVICE;
    h->last_launches = 0;
    if (ap->units.empty()) return MSA_OK;
    if (!contig_k || !contig_v || !pool_k || !pool_v || !block_table || num_blocks < 1) return MSA_ERR_INVALID_ARG;
    if (ap->max_row >= contig_rows || ap->max_bt >= block_table_len) return MSA_ERR_OUT_OF_RANGE;
    if (!aligned16(contig_k) || !aligned16(contig_v) || !aligned16(pool_k) || !aligned16(pool_v) ||
        (reinterpret_cast<uintptr_t>(block_table) & 3u))
        return MSA_ERR_MISALIGNED;
    DeviceGuard guard(h->cfg.device);
    if (guard.err != cudaSuccess) return cuda_fail(guard.err, "msa_kv_append: cudaSetDevice");
    AppendParams ap_params;
    ap_params.units = ap->d_units;
    ap_params.block_table = block_table;
    ap_params.contig_k = contig_k;
    ap_params.contig_v = contig_v;
    ap_params.pool_k = pool_k;
    ap_params.pool_v = pool_v;
    ap_params.row_bytes = static_cast<int64_t>(h->cfg.num_kv_heads) * h->cfg.head_dim * 2;
    ap_params.n_units = static_cast<int32_t>(ap->units.size());
    ap_params.inv_scale = h->kv8 ? h->d_kv8_inv : nullptr;
    ap_params.Hkv = h->cfg.num_kv_heads;
    ap_params.D = h->cfg.head_dim;
    MSA_CUDA(launch_append(ap_params, h->num_sms, static_cast<cudaStream_t>(cuda_stream)));
    h->last_launches = 1;
    return MSA_OK;
}

int msa_check_block_ids(msa_handle h, msa_plan p, msa_append_plan ap, const int32_t *block_table, int64_t block_table_len,
                        int64_t num_blocks, int32_t *device_flag, void *cuda_stream)
{
    if (!h || (!p && !ap) || (p && p->h != h) || (ap && ap->h != h)) return MSA_ERR_INVALID_ARG;
    if (h->planning_only) return MSA_ERR_NO_DEVICE;
    if (!block_table || !device_flag || block_table_len < 0 || num_blocks < 0) return MSA_ERR_INVALID_ARG;
    if ((reinterpret_cast<uintptr_t>(block_table) & 3u) || (reinterpret_cast<uintptr_t>(device_flag) & 3u)) return MSA_ERR_MISALIGNED;
    CheckParams cp;
    memset(&cp, 0, sizeof cp);
    msa_append_plan own = p ? p->wb_append : nullptr;        // fp8 write-back plan: its destinations are an append plan of its own
    if (own && own->max_bt >= block_table_len) return MSA_ERR_OUT_OF_RANGE;
    if (p) {
        const HostPlan &hp = p->hp;
        if (hp.uses_paged && hp.info.max_block_table_index >= block_table_len) return MSA_ERR_OUT_OF_RANGE;
        if (hp.has_writeback && hp.wb_max_bt >= block_table_len) return MSA_ERR_OUT_OF_RANGE;
        cp.vblocks = p->d_vblocks;
        cp.n_vblocks = static_cast<int32_t>(hp.vblocks.size());
        if (hp.has_writeback) {
            cp.vb_dst = p->d_vb_dst;
            cp.n_vb_dst = static_cast<int32_t>(hp.vb_dst.size());
        }
    }
    if (ap) {
        if (ap->max_bt >= block_table_len) return MSA_ERR_OUT_OF_RANGE;
        cp.units = ap->d_units;
        cp.n_units = static_cast<int32_t>(ap->units.size());
    }
    cp.block_table = block_table;
    cp.num_blocks = num_blocks;
    cp.flag = device_flag;
    DeviceGuard guard(h->cfg.device);
    if (guard.err != cudaSuccess) return cuda_fail(guard.err, "msa_check_block_ids: cudaSetDevice");
    MSA_CUDA(launch_check_ids(cp, true, static_cast<cudaStream_t>(cuda_stream)));
    if (own) {
        CheckParams c2;
        memset(&c2, 0, sizeof c2);
        c2.units = own->d_units;
        c2.n_units = static_cast<int32_t>(own->units.size());
        c2.block_table = block_table;
        c2.num_blocks = num_blocks;
        c2.flag = device_flag;
        MSA_CUDA(launch_check_ids(c2, false, static_cast<cudaStream_t>(cuda_stream)));
    }
    return MSA_OK;
}

int msa_last_launch_count(msa_handle h) { return h ? h->last_launches : 0; }

int msa_set_timing(msa_handle h, int max_steps)
{
    if (!h || max_steps < 0) return MSA_ERR_INVALID_ARG;
    if (h->planning_only) return MSA_ERR_NO_DEVICE;
    DeviceGuard guard(h->cfg.device);
    if (guard.err != cudaSuccess) return cuda_fail(guard.err, "msa_set_timing: cudaSetDevice");
    for (cudaEvent_t e : h->ev) cudaEventDestroy(e);
    h->ev.clear();
    h->ev_steps = 0;
    h->timing = max_steps > 0;
    for (int i = 0; i < max_steps * 3; ++i) {
        cudaEvent_t e;
        MSA_CUDA(cudaEventCreate(&e));
        h->ev.push_back(e);
    }
    return MSA_OK;
}

int msa_get_timing(msa_handle h, int32_t *steps, double *fwd_ms_avg, double *merge_ms_avg)
{
    if (!h || !steps || !fwd_ms_avg || !merge_ms_avg) return MSA_ERR_INVALID_ARG;
    *steps = h->ev_steps;
    *fwd_ms_avg = *merge_ms_avg = 0.0;
    if (h->ev_steps == 0) return MSA_OK;
    MSA_CUDA(cudaEventSynchronize(h->ev[static_cast<size_t>(h->ev_steps) * 3 - 1]));
    double a = 0.0, b = 0.0;
    for (int i = 0; i < h->ev_steps; ++i) {
        float f = 0.f, m = 0.f;
        MSA_CUDA(cudaEventElapsedTime(&f, h->ev[i * 3], h->ev[i * 3 + 1]));
        MSA_CUDA(cudaEventElapsedTime(&m, h->ev[i * 3 + 1], h->ev[i * 3 + 2]));
        a += f;
        b += m;
    }
    *fwd_ms_avg = a / h->ev_steps;
    *merge_ms_avg = b / h->ev_steps;
    h->ev_steps = 0;
    return MSA_OK;
}

}  // extern "C"

// ---------------------------------------------------------------------------------------------------------------------------
// msa_forward_static_ws (include/msa.h): msa_forward for callers that cannot allocate the workspace -- an engine that has
// already given all free HBM to its KV pool, or code that may not call cudaMalloc / cudaFree (they synchronise the device)
// while steps are in flight.  The workspace is this array: part of the library's device image, one copy per device, held
// from the moment the CUDA runtime loads this module on a device until the process ends.
//
// In host code `g_static_ws` is only a handle for the symbol, not a device address (handing it to a kernel would fault, or
// quietly touch host memory on a system where the GPU can reach it): the device address comes from
// cudaGetSymbolAddress, looked up once per device with that device current, and that pointer is what the forward and merge
// kernels receive through their parameter structs.
static __device__ __align__(256) unsigned char g_static_ws[MSA_STATIC_WS_BYTES];

namespace {
constexpr int kStaticWsMaxDevices = 64;
std::mutex g_static_ws_mu;
void *g_static_ws_ptr[kStaticWsMaxDevices] = {};     // device address of g_static_ws on device i; NULL = not looked up yet
}  // namespace

extern "C" int msa_forward_static_ws(msa_handle h, msa_plan p, const void *q, int64_t total_q, const void *pool_k,
                                     const void *pool_v, int64_t num_blocks, const int32_t *block_table,
                                     int64_t block_table_len, const void *contig_k, const void *contig_v, int64_t contig_rows,
                                     float softmax_scale, void *o, float *lse, void *cuda_stream)
{
    if (!h || !p || p->h != h) return MSA_ERR_INVALID_ARG;
    if (h->planning_only) return MSA_ERR_NO_DEVICE;
    const int device = h->cfg.device;
    if (device >= kStaticWsMaxDevices) return MSA_ERR_STATIC_WS;
    const size_t need = p->ws_partials + 2 * p->ws_pool + p->ws_ident;
    if (need > static_cast<size_t>(MSA_STATIC_WS_BYTES)) return MSA_ERR_STATIC_WS;      // refused before anything is launched
    void *ws = nullptr;
    {
        DeviceGuard guard(device);      // the symbol's address differs per device: look it up with the handle's device current
        if (guard.err != cudaSuccess) return cuda_fail(guard.err, "msa_forward_static_ws: cudaSetDevice");
        std::lock_guard<std::mutex> lock(g_static_ws_mu);
        if (!g_static_ws_ptr[device]) {
            // one-time set-up on this device (the first call; documented to come before any stream capture)
            void *ptr = nullptr;
            MSA_CUDA(cudaGetSymbolAddress(&ptr, g_static_ws));
            if (!ptr) return MSA_ERR_CUDA;
            g_static_ws_ptr[device] = ptr;
        }
        ws = g_static_ws_ptr[device];
    }
    // (host side of "allocates nothing": msa_create reserved the handle's tensor-map table, a new pointer set appends in place)
    return forward_impl(h, p, q, total_q, pool_k, pool_v, num_blocks, block_table, block_table_len, contig_k, contig_v, contig_rows,
                        softmax_scale, o, lse, ws, static_cast<size_t>(MSA_STATIC_WS_BYTES), cuda_stream, false);
}
