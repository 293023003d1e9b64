// KV write-back (include/msa.h, msa_kv_append): arena rows -> paged cache blocks, 16 tokens per copy unit.
// HBM-bound copy: every byte is read once and written once with 16-byte accesses.
#include "msa_kernels.h"

namespace msa {

__global__ void __launch_bounds__(256) msa_kv_append_kernel(const AppendParams P)
{
    const int64_t row_vec = P.row_bytes / 16;                     // uint4 per token row (Hkv * D * 2 / 16)
    for (int u = blockIdx.x; u < P.n_units; u += gridDim.x) {
        const AppendUnit un = P.units[u];
        const int64_t dst_row = static_cast<int64_t>(__ldg(P.block_table + un.bt_index)) * kBlock;
        const int64_t n = un.nvalid * row_vec;
        const uint4 *sk = reinterpret_cast<const uint4 *>(P.contig_k) + un.src_row * row_vec;
        const uint4 *sv = reinterpret_cast<const uint4 *>(P.contig_v) + un.src_row * row_vec;
        uint4 *dk = reinterpret_cast<uint4 *>(P.pool_k) + dst_row * row_vec;
        uint4 *dv = reinterpret_cast<uint4 *>(P.pool_v) + dst_row * row_vec;
        for (int64_t i = threadIdx.x; i < n; i += blockDim.x) {
            const uint4 a = __ldg(sk + i), b = __ldg(sv + i);
            dk[i] = a;
            dv[i] = b;
        }
    }
}

cudaError_t launch_append(const AppendParams &p, int num_sms, cudaStream_t stream)
{
    if (p.n_units <= 0) return cudaSuccess;
    const int grid = p.n_units < num_sms * 8 ? p.n_units : num_sms * 8;
    msa_kv_append_kernel<<<grid, 256, 0, stream>>>(p);
    return cudaGetLastError();
}

}  // namespace msa
