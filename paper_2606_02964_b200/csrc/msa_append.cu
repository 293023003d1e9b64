// KV write-back (include/msa.h, msa_kv_append): arena rows -> paged cache blocks, 16 tokens per copy unit.
// HBM-bound copy: every byte is read once and written once with 16-byte accesses.  One copy unit is 16 tokens x
// (Hkv*D*2) bytes for each of K and V -- contiguous on both sides -- so a block walks its unit in chunks of
// kInFlight x 16 bytes per thread and tensor: all loads of a chunk are issued before the first store (the copy is
// latency-bound otherwise: a 64 KB unit is only a handful of trips per thread).
#include "msa_kernels.h"

namespace msa {

constexpr int kAppendThreads = 256;
constexpr int kInFlight = 4;          // uint4 per thread, tensor and trip

__global__ void __launch_bounds__(kAppendThreads) msa_kv_append_kernel(const AppendParams P)
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
        for (int64_t base = 0; base < n; base += kAppendThreads * kInFlight) {
            uint4 a[kInFlight], b[kInFlight];
#pragma unroll
            for (int j = 0; j < kInFlight; ++j) {
                const int64_t i = base + j * kAppendThreads + threadIdx.x;
                if (i < n) {
                    a[j] = __ldcs(sk + i);                         // streaming: read once
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

cudaError_t launch_append(const AppendParams &p, int num_sms, cudaStream_t stream)
{
    if (p.n_units <= 0) return cudaSuccess;
    const int grid = p.n_units < num_sms * 8 ? p.n_units : num_sms * 8;
    msa_kv_append_kernel<<<grid, kAppendThreads, 0, stream>>>(p);
    return cudaGetLastError();
}

}  // namespace msa
