// LSE-merge kernel: combines the split-KV partials of one work item.
//   LSE = ln sum_s exp(LSE_s),   O = sum_s exp(LSE_s - LSE) * O_s      (fixed split order:
// deterministic, no float atomics).  One CTA per split item, one warp per packed row.
#include <cuda_bf16.h>
#include <math.h>

#include "msa_kernels.h"

namespace msa {

template <int D>
__global__ void __launch_bounds__(128) msa_merge_kernel(const MergeParams P)
{
    const MergeItem it = P.items[blockIdx.x];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int rows = it.n_tok * P.G;
    constexpr int E = D / 32;   // floats per lane
    for (int row = warp; row < rows; row += blockDim.x >> 5) {
        const int g = row / it.n_tok, t = row - g * it.n_tok;
        const int head = P.kv_to_q[it.kvh * P.G + g];
        float mx = -INFINITY;
        for (int s = 0; s < it.n_partials; ++s) {
            const float *part = P.workspace + it.first_off + s * it.stride;
            mx = fmaxf(mx, part[static_cast<size_t>(rows) * D + row]);
        }
        float acc[E];
#pragma unroll
        for (int e = 0; e < E; ++e) acc[e] = 0.f;
        float lse = -INFINITY;
        if (mx > -INFINITY) {
            float sum = 0.f;
            for (int s = 0; s < it.n_partials; ++s) {
                const float *part = P.workspace + it.first_off + s * it.stride;
                sum += expf(part[static_cast<size_t>(rows) * D + row] - mx);
            }
            lse = mx + logf(sum);
            for (int s = 0; s < it.n_partials; ++s) {
                const float *part = P.workspace + it.first_off + s * it.stride;
                const float w = expf(part[static_cast<size_t>(rows) * D + row] - lse);
                const float *orow = part + static_cast<size_t>(row) * D + lane * E;
#pragma unroll
                for (int e = 0; e < E; ++e) acc[e] = fmaf(w, orow[e], acc[e]);
            }
        }
        __nv_bfloat16 *dst = reinterpret_cast<__nv_bfloat16 *>(P.o) +
                             (static_cast<size_t>(it.q_row0 + t) * P.Hq + head) * D + lane * E;
#pragma unroll
        for (int e = 0; e < E; e += 2)
            *reinterpret_cast<__nv_bfloat162 *>(dst + e) = __floats2bfloat162_rn(acc[e], acc[e + 1]);
        if (lane == 0) P.lse[static_cast<size_t>(it.q_row0 + t) * P.Hq + head] = lse;
    }
}

cudaError_t launch_merge(const MergeParams &p, int n_items, cudaStream_t stream)
{
    if (n_items <= 0) return cudaSuccess;
    if (p.D == 128)
        msa_merge_kernel<128><<<n_items, 128, 0, stream>>>(p);
    else
        msa_merge_kernel<64><<<n_items, 128, 0, stream>>>(p);
    return cudaGetLastError();
}

}  // namespace msa
