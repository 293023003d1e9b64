// LSE-merge kernel: combines the split-KV partials of one work item.
//   LSE = ln sum_s exp(LSE_s),   O = sum_s exp(LSE_s - LSE) * O_s      (fixed split order:
// deterministic, no float atomics).  grid = (split items, row blocks); one warp per packed
// row, each lane owns D/32 consecutive output elements.
#include <cuda_bf16.h>
#include <math.h>

#include "msa_kernels.h"

namespace msa {

constexpr int kMergeWarps = 8;

template <int D>
__global__ void __launch_bounds__(kMergeWarps * 32) msa_merge_kernel(const MergeParams P)
{
    const MergeItem it = P.items[blockIdx.x];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int rows = it.n_tok * P.G;
    const int row = blockIdx.y * kMergeWarps + warp;
    if (row >= rows) return;
    constexpr int E = D / 32;   // floats per lane
    const int g = row / it.n_tok, t = row - g * it.n_tok;
    const int head = P.kv_to_q[it.kvh * P.G + g];
    const float *base = P.workspace + it.first_off;
    // lane s holds LSE_s (n_partials <= 32 in practice; loop covers more)
    float mx = -INFINITY;
    for (int s = lane; s < it.n_partials; s += 32) mx = fmaxf(mx, base[s * it.stride + static_cast<size_t>(rows) * D + row]);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, o));
    float acc[E];
#pragma unroll
    for (int e = 0; e < E; ++e) acc[e] = 0.f;
    float lse = -INFINITY;
    if (mx > -INFINITY) {
        float sum = 0.f;
        for (int s = 0; s < it.n_partials; ++s) sum += expf(base[s * it.stride + static_cast<size_t>(rows) * D + row] - mx);
        lse = mx + logf(sum);
        for (int s = 0; s < it.n_partials; ++s) {
            const float *part = base + s * it.stride;
            const float w = expf(part[static_cast<size_t>(rows) * D + row] - lse);
            const float *orow = part + static_cast<size_t>(row) * D + lane * E;
            if (E == 4) {
                const float4 v = *reinterpret_cast<const float4 *>(orow);
                acc[0] = fmaf(w, v.x, acc[0]);
                acc[1] = fmaf(w, v.y, acc[1]);
                acc[2] = fmaf(w, v.z, acc[2]);
                acc[3] = fmaf(w, v.w, acc[3]);
            } else {
                const float2 v = *reinterpret_cast<const float2 *>(orow);
                acc[0] = fmaf(w, v.x, acc[0]);
                acc[1] = fmaf(w, v.y, acc[1]);
            }
        }
    }
    __nv_bfloat16 *dst = reinterpret_cast<__nv_bfloat16 *>(P.o) + (static_cast<size_t>(it.q_row0 + t) * P.Hq + head) * D + lane * E;
#pragma unroll
    for (int e = 0; e < E; e += 2)
        *reinterpret_cast<__nv_bfloat162 *>(dst + e) = __floats2bfloat162_rn(acc[e], acc[e + 1]);
    if (lane == 0) P.lse[static_cast<size_t>(it.q_row0 + t) * P.Hq + head] = lse;
}

cudaError_t launch_merge(const MergeParams &p, int n_items, int max_rows, cudaStream_t stream)
{
    if (n_items <= 0 || max_rows <= 0) return cudaSuccess;
    dim3 grid(n_items, (max_rows + kMergeWarps - 1) / kMergeWarps);
    if (p.D == 128)
        msa_merge_kernel<128><<<grid, kMergeWarps * 32, 0, stream>>>(p);
    else
        msa_merge_kernel<64><<<grid, kMergeWarps * 32, 0, stream>>>(p);
    return cudaGetLastError();
}

}  // namespace msa
