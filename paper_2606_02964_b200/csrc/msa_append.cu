// KV write-back as its own launch (include/msa.h, msa_kv_append): arena rows -> paged cache blocks, 16 tokens per copy
// unit.  HBM-bound copy: every byte is read once and written once.  A copy unit is contiguous on both sides (up to
// 16 rows x Hkv*D*2 bytes per tensor), so each persistent CTA moves whole units with the bulk-copy engine:
// cp.async.bulk global -> shared (mbarrier completion), then shared -> global (bulk async-group), kStages units in flight.
// One thread per CTA issues everything; the SM's other resources stay idle.
#include "msa_kernels.h"
#include "msa_ptx.cuh"

namespace msa {

constexpr int kAppendStages = 3;
constexpr int kAppendMaxUnitBytes = 2 * 16 * 2048;     // K + V of one unit at Hkv*D*2 <= 2048 bytes per row (else the fallback kernel)

__global__ void __launch_bounds__(32) msa_kv_append_bulk_kernel(const AppendParams P)
{
    extern __shared__ __align__(128) uint8_t smem[];
    __shared__ uint64_t full[kAppendStages];
    if (threadIdx.x != 0) return;
    const uint32_t rb = static_cast<uint32_t>(P.row_bytes);
    const uint32_t stage_bytes = 2u * 16u * rb;
    for (int s = 0; s < kAppendStages; ++s) mbar_init(smem_u32(&full[s]), 1);
    fence_mbar_init();
    const int first = blockIdx.x, stride = gridDim.x;
    const int n_mine = first < P.n_units ? (P.n_units - first + stride - 1) / stride : 0;
    auto load = [&](int i) {          // i-th unit of this CTA -> stage i % kAppendStages
        const int s = i % kAppendStages;
        const AppendUnit un = P.units[first + i * stride];
        const uint32_t bytes = static_cast<uint32_t>(un.nvalid) * rb;
        const uint32_t dst = smem_u32(smem) + s * stage_bytes, bar = smem_u32(&full[s]);
        const uint8_t *sk = static_cast<const uint8_t *>(P.contig_k) + un.src_row * P.row_bytes;
        const uint8_t *sv = static_cast<const uint8_t *>(P.contig_v) + un.src_row * P.row_bytes;
        mbar_arrive_expect_tx(bar, 2u * bytes);
        asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                     ::"r"(dst), "l"(sk), "r"(bytes), "r"(bar) : "memory");
        asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                     ::"r"(dst + 16u * rb), "l"(sv), "r"(bytes), "r"(bar) : "memory");
    };
    for (int i = 0; i < n_mine && i < kAppendStages - 1; ++i) load(i);
    for (int i = 0; i < n_mine; ++i) {
        const int s = i % kAppendStages;
        // the stage that unit i + kStages - 1 will use was stored from by unit i - 1: its stores must have read it
        if (i + kAppendStages - 1 < n_mine) {
            asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
            load(i + kAppendStages - 1);
        }
        mbar_wait(smem_u32(&full[s]), static_cast<uint32_t>(i / kAppendStages) & 1u);
        const AppendUnit un = P.units[first + i * stride];
        const uint32_t bytes = static_cast<uint32_t>(un.nvalid) * rb;
        const int64_t dst_row = static_cast<int64_t>(__ldg(P.block_table + un.bt_index)) * kBlock;
        uint8_t *dk = static_cast<uint8_t *>(P.pool_k) + dst_row * P.row_bytes;
        uint8_t *dv = static_cast<uint8_t *>(P.pool_v) + dst_row * P.row_bytes;
        const uint32_t src = smem_u32(smem) + s * stage_bytes;
        asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(dk), "r"(src), "r"(bytes) : "memory");
        asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(dv), "r"(src + 16u * rb), "r"(bytes) : "memory");
        asm volatile("cp.async.bulk.commit_group;" ::: "memory");
    }
    asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");
}

// Fallback for rows wider than 2 KB: 16-byte loads and stores, 8 loads in flight per thread before the first store.
constexpr int kAppendThreads = 256;
constexpr int kInFlight = 4;

__global__ void __launch_bounds__(kAppendThreads) msa_kv_append_kernel(const AppendParams P)
{
    const int64_t row_vec = P.row_bytes / 16;
    for (int u = blockIdx.x; u < P.n_units; u += gridDim.x) {
        const AppendUnit un = P.units[u];
        const int64_t dst_row = static_cast<int64_t>(__ldg(P.block_table + un.bt_index)) * kBlock;
        const int64_t n = un.nvalid * row_vec;
        const uint4 *sk = reinterpret_cast<const uint4 *>(P.contig_k) + un.src_row * row_vec;
        const uint4 *sv = reinterpret_cast<const uint4 *>(P.contig_v) + un.src_row * row_vec;
        uint4 *dk = reinterpret_cast<uint4 *>(P.pool_k) + dst_row * row_vec;
        uint4 *dv = reinterpret_cast<uint4 *>(P.pool_v) + dst_row * row_vec;
        for (int64_t base = 0; base < n; base += kAppendThreads * kInFlight) {
            uint4 a[kInFlight], b[kInFlight];
#pragma unroll
            for (int j = 0; j < kInFlight; ++j) {
                const int64_t i = base + j * kAppendThreads + threadIdx.x;
                if (i < n) {
                    a[j] = __ldcs(sk + i);
                    b[j] = __ldcs(sv + i);
                }
            }
#pragma unroll
            for (int j = 0; j < kInFlight; ++j) {
                const int64_t i = base + j * kAppendThreads + threadIdx.x;
                if (i < n) {
                    dk[i] = a[j];
                    dv[i] = b[j];
                }
            }
        }
    }
}

// fp8 (E4M3) pool: the rows are quantised on the way -- code = E4M3 code nearest to value / scale, ties to even, values
// beyond +-448 saturate, NaN gives the NaN code (cvt.rn.satfinite.e4m3x2.f32).  1 / scale is a power of two, so the
// division is exact.  HBM-bound: 2 bytes read and 1 written per element; a thread turns 16 bf16 (32 B) into 16 codes.
__device__ __forceinline__ uint32_t quant4_e4m3(uint32_t lo2, uint32_t hi2, float inv)
{
    const float f0 = __uint_as_float(lo2 << 16) * inv, f1 = __uint_as_float(lo2 & 0xffff0000u) * inv;
    const float f2 = __uint_as_float(hi2 << 16) * inv, f3 = __uint_as_float(hi2 & 0xffff0000u) * inv;
    uint16_t a, b;
    asm("cvt.rn.satfinite.e4m3x2.f32 %0, %1, %2;" : "=h"(a) : "f"(f1), "f"(f0));
    asm("cvt.rn.satfinite.e4m3x2.f32 %0, %1, %2;" : "=h"(b) : "f"(f3), "f"(f2));
    return static_cast<uint32_t>(a) | (static_cast<uint32_t>(b) << 16);
}

__global__ void __launch_bounds__(kAppendThreads) msa_kv_append_q8_kernel(const AppendParams P)
{
    const int64_t row_elems = P.row_bytes / 2;          // Hkv * D
    const int64_t row_chunks = row_elems / 16;          // 16-element chunks per row (D is a multiple of 16)
    const int chunks_per_head = P.D / 16;
    for (int u = blockIdx.x; u < P.n_units; u += gridDim.x) {
        const AppendUnit un = P.units[u];
        const int64_t dst_row = static_cast<int64_t>(__ldg(P.block_table + un.bt_index)) * kBlock;
        const int64_t n = un.nvalid * row_chunks;
        const uint4 *sk = reinterpret_cast<const uint4 *>(P.contig_k) + un.src_row * row_chunks * 2;
        const uint4 *sv = reinterpret_cast<const uint4 *>(P.contig_v) + un.src_row * row_chunks * 2;
        uint4 *dk = reinterpret_cast<uint4 *>(P.pool_k) + dst_row * row_chunks;
        uint4 *dv = reinterpret_cast<uint4 *>(P.pool_v) + dst_row * row_chunks;
        for (int64_t i = threadIdx.x; i < n; i += kAppendThreads) {
            const int kvh = static_cast<int>((i % row_chunks) / chunks_per_head);
            const float ik = __ldg(P.inv_scale + kvh), iv = __ldg(P.inv_scale + P.Hkv + kvh);
            const uint4 k0 = __ldcs(sk + 2 * i), k1 = __ldcs(sk + 2 * i + 1);
            const uint4 v0 = __ldcs(sv + 2 * i), v1 = __ldcs(sv + 2 * i + 1);
            dk[i] = make_uint4(quant4_e4m3(k0.x, k0.y, ik), quant4_e4m3(k0.z, k0.w, ik), quant4_e4m3(k1.x, k1.y, ik),
                               quant4_e4m3(k1.z, k1.w, ik));
            dv[i] = make_uint4(quant4_e4m3(v0.x, v0.y, iv), quant4_e4m3(v0.z, v0.w, iv), quant4_e4m3(v1.x, v1.y, iv),
                               quant4_e4m3(v1.z, v1.w, iv));
        }
    }
}

cudaError_t configure_append()
{
    return cudaFuncSetAttribute(msa_kv_append_bulk_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                kAppendStages * kAppendMaxUnitBytes);
}

cudaError_t launch_append(const AppendParams &p, int num_sms, cudaStream_t stream)
{
    if (p.n_units <= 0) return cudaSuccess;
    if (p.inv_scale != nullptr) {
        const int grid = p.n_units < num_sms * 8 ? p.n_units : num_sms * 8;
        msa_kv_append_q8_kernel<<<grid, kAppendThreads, 0, stream>>>(p);
        return cudaGetLastError();
    }
    if (2 * 16 * p.row_bytes <= kAppendMaxUnitBytes) {
        const int grid = p.n_units < num_sms ? p.n_units : num_sms;
        msa_kv_append_bulk_kernel<<<grid, 32, kAppendStages * 2 * 16 * static_cast<size_t>(p.row_bytes), stream>>>(p);
    } else {
        const int grid = p.n_units < num_sms * 8 ? p.n_units : num_sms * 8;
        msa_kv_append_kernel<<<grid, kAppendThreads, 0, stream>>>(p);
    }
    return cudaGetLastError();
}

}  // namespace msa
