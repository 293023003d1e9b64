// fp8 (E4M3) pool, launches with prefill (pair-mode) units: dequantising pre-pass.
//
// A prefill launch reads every cached K/V tile once per q-tile group of its (run, KV head) -- cfg2: eight times, from L2 --
// and converting the codes inside the forward kernel would repeat the conversion as often, on the four warps that are not
// exponentiating (the conversion, not HBM, is what bounds the fp8 variant).  So for such a launch the
// cached blocks the plan refers to are converted ONCE, into a compact bf16 copy in the caller's workspace (block j of the
// copy = the j-th distinct block-table entry of the plan), and the bf16 forward kernel runs on that copy with an identity
// block table.  HBM-bound: one byte read and two written per element.  Short-query launches (no reuse: every byte is read
// once) keep the codes all the way into shared memory (msa_fwd_pipe_kernel<D, true, 1>).
#include "msa_kernels.h"
#include "msa_kv8.cuh"

namespace msa {

constexpr int kDequantThreads = 256;

__global__ void __launch_bounds__(kDequantThreads) msa_kv8_dequant_kernel(const DequantParams P)
{
    const int chunks_per_row = P.Hkv * P.D / 16;              // 16 codes per thread and step
    const int chunks_per_head = P.D / 16;
    const int chunks = kBlock * chunks_per_row;
    for (int j = blockIdx.x; j < P.n_blocks; j += gridDim.x) {
        const int64_t src_blk = __ldg(P.block_table + __ldg(P.src_bt + j));
        if (threadIdx.x == 0) P.ident[j] = j;
        const uint4 *sk = reinterpret_cast<const uint4 *>(P.pool_k) + src_blk * chunks;
        const uint4 *sv = reinterpret_cast<const uint4 *>(P.pool_v) + src_blk * chunks;
        uint4 *dk = reinterpret_cast<uint4 *>(P.out_k) + static_cast<int64_t>(j) * chunks * 2;
        uint4 *dv = reinterpret_cast<uint4 *>(P.out_v) + static_cast<int64_t>(j) * chunks * 2;
        for (int i = threadIdx.x; i < chunks; i += kDequantThreads) {
            const int kvh = (i % chunks_per_row) / chunks_per_head;
            const uint32_t mk = __ldg(P.kv8_mul + kvh), mv = __ldg(P.kv8_mul + P.Hkv + kvh);
            const uint4 k = __ldcs(sk + i), v = __ldcs(sv + i);
            dk[2 * i] = make_uint4(e4m3x2_to_bf16x2(k.x, mk), e4m3x2_to_bf16x2(k.x >> 16, mk), e4m3x2_to_bf16x2(k.y, mk),
                                   e4m3x2_to_bf16x2(k.y >> 16, mk));
            dk[2 * i + 1] = make_uint4(e4m3x2_to_bf16x2(k.z, mk), e4m3x2_to_bf16x2(k.z >> 16, mk), e4m3x2_to_bf16x2(k.w, mk),
                                       e4m3x2_to_bf16x2(k.w >> 16, mk));
            dv[2 * i] = make_uint4(e4m3x2_to_bf16x2(v.x, mv), e4m3x2_to_bf16x2(v.x >> 16, mv), e4m3x2_to_bf16x2(v.y, mv),
                                   e4m3x2_to_bf16x2(v.y >> 16, mv));
            dv[2 * i + 1] = make_uint4(e4m3x2_to_bf16x2(v.z, mv), e4m3x2_to_bf16x2(v.z >> 16, mv), e4m3x2_to_bf16x2(v.w, mv),
                                       e4m3x2_to_bf16x2(v.w >> 16, mv));
        }
    }
}

cudaError_t launch_dequant(const DequantParams &p, int num_sms, cudaStream_t stream)
{
    if (p.n_blocks <= 0) return cudaSuccess;
    const int grid = p.n_blocks < num_sms * 8 ? p.n_blocks : num_sms * 8;
    msa_kv8_dequant_kernel<<<grid, kDequantThreads, 0, stream>>>(p);
    return cudaGetLastError();
}

}  // namespace msa
