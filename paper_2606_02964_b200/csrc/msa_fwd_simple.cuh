// msa_fwd_simple: the straight-line MSA forward kernel (debug / bring-up variant).
//
// One CTA of 128 threads walks its work units; every phase is separated by a CTA barrier:
//   TMA (Q once; per KV tile 8 virtual blocks of K and V, paged or contiguous through the
//   same 64x16 box) -> tcgen05.mma S = Q K^T (TMEM) -> one thread per packed row: mask by
//   absolute position, online softmax, P (bf16) back to TMEM, rescale O -> tcgen05.mma
//   O += P V (A from TMEM, V MN-major from smem) -> epilogue.
// No overlap at all: it exists to validate descriptors, layouts and masking, and as the
// on-device cross-check for the pipelined kernel (env MSA_KERNEL=simple).
#pragma once
#include <math.h>

#include "msa_kernels.h"
#include "msa_ptx.cuh"

namespace msa {

template <int D>
struct SimpleCfg {
    static constexpr int kHalves = D / 64;
    static constexpr int kHalfBytes = kTileM * 128;            // 128 rows x 128 B (64 bf16)
    static constexpr int kTileBytes = kHalves * kHalfBytes;
    static constexpr int kSmemBytes = 3 * kTileBytes + 1024;   // Q, K, V + alignment slack
    static constexpr uint32_t kColS = 0, kColP = 128, kColO = 256;
};

template <int D>
__global__ void __launch_bounds__(128, 1) msa_fwd_simple_kernel(const __grid_constant__ FwdParams P)
{
    using C = SimpleCfg<D>;
    extern __shared__ uint8_t smem_raw[];
    __shared__ __align__(8) uint64_t s_bar[2];
    __shared__ uint32_t s_tmem;
    __shared__ VBlock s_vb[kVbPerTile];

    const uint32_t raw = smem_u32(smem_raw);
    const uint32_t base = (raw + 1023u) & ~1023u;
    const uint32_t sQ = base, sK = base + C::kTileBytes, sV = base + 2 * C::kTileBytes;
    uint8_t *gV = smem_raw + (sV - raw);
    const uint32_t bar_load = smem_u32(&s_bar[0]), bar_mma = smem_u32(&s_bar[1]);
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;

    if (warp == 0) {
        tmem_alloc(smem_u32(&s_tmem), 512);
        tmem_relinquish();
    }
    if (tid == 32) {
        mbar_init(bar_load, 1);
        mbar_init(bar_mma, 1);
        fence_mbar_init();
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = s_tmem;
    const uint32_t trow = tmem + (static_cast<uint32_t>(warp * 32) << 16);
    uint32_t ph_load = 0, ph_mma = 0;
    const int G = P.G, R = P.R;
    const float sl = P.scale_log2;
    constexpr uint32_t idesc_s = make_idesc(128, 128, false);
    constexpr uint32_t idesc_o = make_idesc(128, D, true);

    for (int u = P.cta_unit_begin[blockIdx.x]; u < P.cta_unit_begin[blockIdx.x + 1]; ++u) {
        const WorkUnit wu = P.units[u];
        const int g = tid / R, t = tid - g * R;
        const bool row_valid = (g < G) && (t < wu.n_tok);
        const int p_row = wu.q_abs0 + t;
        const int head = row_valid ? P.kv_to_q[wu.kvh * G + g] : 0;
        float m = -INFINITY, l = 0.f;
        const bool has_tiles = wu.tile_end > wu.tile_begin;

        if (has_tiles) {
            if (warp == 0) {
                if (lane == 0) mbar_arrive_expect_tx(bar_load, static_cast<uint32_t>(G * R * D * 2));
                __syncwarp();
                if (lane < G) {
                    const int hq = P.kv_to_q[wu.kvh * G + lane];
#pragma unroll
                    for (int h = 0; h < C::kHalves; ++h)
                        tma_load_2d(sQ + h * C::kHalfBytes + lane * R * 128, &P.tm_q, bar_load, hq * D + h * 64,
                                    wu.q_row0);
                }
            }
            mbar_wait(bar_load, ph_load);
            ph_load ^= 1;
        }

        for (int tile = wu.tile_begin; tile < wu.tile_end; ++tile) {
            const int nvb = min(kVbPerTile, wu.vb_count - tile * kVbPerTile);
            if (tid < kVbPerTile) {
                VBlock vb = {0, 0, 0, 0};
                if (tid < nvb) vb = P.vblocks[wu.vb_begin + tile * kVbPerTile + tid];
                s_vb[tid] = vb;
                if (tid == 0) mbar_arrive_expect_tx(bar_load, static_cast<uint32_t>(nvb * 2 * kBlock * D * 2));   // nvb counts real blocks only
                if (tid < nvb && vb.nvalid > 0) {
                    const void *tk = vb.paged ? &P.tm_pool_k[0] : &P.tm_ctg_k[0];
                    const void *tv = vb.paged ? &P.tm_pool_v[0] : &P.tm_ctg_v[0];
                    const int row = vb.paged ? P.block_table[vb.src] * kBlock : vb.src;
#pragma unroll
                    for (int h = 0; h < C::kHalves; ++h) {
                        tma_load_2d(sK + h * C::kHalfBytes + tid * (kBlock * 128), tk, bar_load, wu.kvh * D + h * 64, row);
                        tma_load_2d(sV + h * C::kHalfBytes + tid * (kBlock * 128), tv, bar_load, wu.kvh * D + h * 64, row);
                    }
                }
            }
            __syncthreads();
            mbar_wait(bar_load, ph_load);
            ph_load ^= 1;

            bool ragged = false;
            int tile_max_abs = -1;
#pragma unroll
            for (int b = 0; b < kVbPerTile; ++b) {
                ragged |= s_vb[b].nvalid < kBlock;
                if (s_vb[b].nvalid > 0) tile_max_abs = max(tile_max_abs, s_vb[b].abs_start + s_vb[b].nvalid - 1);
            }
            if (ragged) {
                // P is 0 on invalid slots, but 0 * NaN = NaN: the V rows of invalid slots
                // (block tails, missing blocks) must hold zeros before the PV MMA reads them.
                if ((tid & 15) >= s_vb[tid >> 4].nvalid) {
#pragma unroll
                    for (int h = 0; h < C::kHalves; ++h) {
                        uint4 *rowp = reinterpret_cast<uint4 *>(gV + h * C::kHalfBytes + tid * 128);
#pragma unroll
                        for (int i = 0; i < 8; ++i) rowp[i] = make_uint4(0, 0, 0, 0);
                    }
                }
                fence_proxy_async_smem();
            }
            __syncthreads();
            if (tid == 0) {
                tc_fence_after();
#pragma unroll
                for (int k = 0; k < D / 16; ++k) {
                    const uint32_t off = (k >> 2) * C::kHalfBytes + (k & 3) * 32;
                    umma_ss(tmem + C::kColS, make_smem_desc(sQ + off, 16, 1024), make_smem_desc(sK + off, 16, 1024),
                            idesc_s, k > 0);
                }
                umma_commit(bar_mma);
            }
            mbar_wait(bar_mma, ph_mma);
            ph_mma ^= 1;
            tc_fence_after();

            // ---- softmax on my row ------------------------------------------------
            uint32_t sr[128];
#pragma unroll
            for (int c = 0; c < 4; ++c) tmem_ld32(trow + C::kColS + c * 32, *reinterpret_cast<uint32_t(*)[32]>(&sr[c * 32]));
            tmem_wait_ld();
            const bool need_mask = ragged || tile_max_abs > wu.q_abs0;
            if (need_mask) {
#pragma unroll
                for (int b = 0; b < kVbPerTile; ++b) {
                    const int lim = min(s_vb[b].nvalid, p_row - s_vb[b].abs_start + 1);
#pragma unroll
                    for (int j = 0; j < kBlock; ++j)
                        if (j >= lim) sr[b * kBlock + j] = 0xff800000u;   // -inf
                }
            }
            float mx = -INFINITY;
#pragma unroll
            for (int j = 0; j < 128; ++j) mx = fmaxf(mx, __uint_as_float(sr[j]));
            const float m_new = fmaxf(m, mx);
            const float m_use = (m_new == -INFINITY) ? 0.f : m_new;
            const float alpha = (m == m_new) ? 1.f : ex2_approx((m - m_new) * sl);
            const float neg_ms = -m_use * sl;
            float rowsum = 0.f;
#pragma unroll
            for (int c = 0; c < 8; ++c) {
                uint32_t pk[16];
#pragma unroll
                for (int j = 0; j < 8; ++j) {
                    const float p0 = ex2_approx(fmaf(__uint_as_float(sr[c * 16 + 2 * j]), sl, neg_ms));
                    const float p1 = ex2_approx(fmaf(__uint_as_float(sr[c * 16 + 2 * j + 1]), sl, neg_ms));
                    rowsum += p0 + p1;
                    pk[j] = pack_bf16x2(p0, p1);
                }
#pragma unroll
                for (int j = 0; j < 8; ++j) sr[c * 8 + j] = pk[j];   // reuse sr[0..63] as the packed P row
            }
            l = l * alpha + rowsum;
            m = m_new;
#pragma unroll
            for (int c = 0; c < 4; ++c)
                tmem_st16(trow + C::kColP + c * 16, *reinterpret_cast<uint32_t(*)[16]>(&sr[c * 16]));
            if (tile > wu.tile_begin && __any_sync(0xffffffffu, alpha != 1.f)) {
#pragma unroll
                for (int c = 0; c < D / 32; ++c) {
                    uint32_t orr[32];
                    tmem_ld32(trow + C::kColO + c * 32, orr);
                    tmem_wait_ld();
#pragma unroll
                    for (int j = 0; j < 32; ++j) orr[j] = __float_as_uint(__uint_as_float(orr[j]) * alpha);
                    tmem_st32(trow + C::kColO + c * 32, orr);
                }
            }
            tmem_wait_st();
            tc_fence_before();
            __syncthreads();
            if (tid == 0) {
                tc_fence_after();
#pragma unroll
                for (int k = 0; k < kTileN / 16; ++k)
                    umma_ts(tmem + C::kColO, tmem + C::kColP + k * 8,
                            make_smem_desc(sV + k * (kBlock * 128), C::kHalfBytes, 1024), idesc_o,
                            (tile > wu.tile_begin || k > 0) ? 1u : 0u);
                umma_commit(bar_mma);
            }
            mbar_wait(bar_mma, ph_mma);
            ph_mma ^= 1;
            tc_fence_after();
        }

        // ---- epilogue -------------------------------------------------------------
        const float inv_l = (l > 0.f) ? 1.f / l : 0.f;
        const float lse_val = (l > 0.f) ? (m * sl + log2f(l)) * 0.6931471805599453f : -INFINITY;
        const int rows = wu.n_tok * G;
        if (wu.partial_off < 0) {
            __nv_bfloat16 *orow =
                reinterpret_cast<__nv_bfloat16 *>(P.o) + (static_cast<size_t>(wu.q_row0 + t) * P.Hq + head) * D;
#pragma unroll
            for (int c = 0; c < D / 32; ++c) {
                uint32_t orr[32];
                if (has_tiles) {
                    tmem_ld32(trow + C::kColO + c * 32, orr);
                    tmem_wait_ld();
                } else {
#pragma unroll
                    for (int j = 0; j < 32; ++j) orr[j] = 0;
                }
                if (row_valid) {
#pragma unroll
                    for (int j = 0; j < 4; ++j) {
                        uint4 v;
                        v.x = pack_bf16x2(__uint_as_float(orr[8 * j + 0]) * inv_l, __uint_as_float(orr[8 * j + 1]) * inv_l);
                        v.y = pack_bf16x2(__uint_as_float(orr[8 * j + 2]) * inv_l, __uint_as_float(orr[8 * j + 3]) * inv_l);
                        v.z = pack_bf16x2(__uint_as_float(orr[8 * j + 4]) * inv_l, __uint_as_float(orr[8 * j + 5]) * inv_l);
                        v.w = pack_bf16x2(__uint_as_float(orr[8 * j + 6]) * inv_l, __uint_as_float(orr[8 * j + 7]) * inv_l);
                        *reinterpret_cast<uint4 *>(orow + c * 32 + j * 8) = v;
                    }
                }
            }
            if (row_valid) P.lse[static_cast<size_t>(wu.q_row0 + t) * P.Hq + head] = lse_val;
        } else {
            float *part = P.workspace + wu.partial_off;
            const int prow = g * wu.n_tok + t;
#pragma unroll
            for (int c = 0; c < D / 32; ++c) {
                uint32_t orr[32];
                if (has_tiles) {
                    tmem_ld32(trow + C::kColO + c * 32, orr);
                    tmem_wait_ld();
                } else {
#pragma unroll
                    for (int j = 0; j < 32; ++j) orr[j] = 0;
                }
                if (row_valid) {
#pragma unroll
                    for (int j = 0; j < 8; ++j) {
                        float4 v = make_float4(__uint_as_float(orr[4 * j + 0]) * inv_l, __uint_as_float(orr[4 * j + 1]) * inv_l,
                                               __uint_as_float(orr[4 * j + 2]) * inv_l, __uint_as_float(orr[4 * j + 3]) * inv_l);
                        *reinterpret_cast<float4 *>(part + static_cast<size_t>(prow) * D + c * 32 + j * 4) = v;
                    }
                }
            }
            if (row_valid) part[static_cast<size_t>(rows) * D + prow] = lse_val;
        }
        tc_fence_before();
        __syncthreads();
    }

    if (warp == 0) tmem_dealloc(tmem, 512);
}

}  // namespace msa
