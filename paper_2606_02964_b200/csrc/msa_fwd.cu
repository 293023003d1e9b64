// Forward-kernel launcher for libmsa (sm_100a only).
#include "msa_fwd_pipe.cuh"

namespace msa {

template <int D, bool KV8, int QT>
static cudaError_t configure_one()
{
    return cudaFuncSetAttribute(msa_fwd_pipe_kernel<D, KV8, QT>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                PipeCfg<D, KV8, QT>::kSmemBytes);
}

template <int D, bool KV8, int QT>
static void launch_one(const FwdParams &p, int num_ctas, cudaStream_t stream)
{
    msa_fwd_pipe_kernel<D, KV8, QT><<<num_ctas, 512, PipeCfg<D, KV8, QT>::kSmemBytes, stream>>>(p);
}

// The kernel needs more dynamic shared memory than the default limit; the attribute is per device and
// per function, so the handle sets it once for its own device (msa_create).  A handle with an fp8 pool uses three
// kernels: the fp8 variant in its two shared-memory layouts (room for the two Q tiles of pair-mode units, or -- short
// queries only -- one Q tile and a deeper staging ring), and the bf16 kernel behind the dequantising pre-pass for
// launches that load their cached tiles several times (msa_dequant.cu).
cudaError_t configure_fwd(int head_dim, bool kv8)
{
    cudaError_t e = head_dim == 128 ? configure_one<128, false, 2>() : configure_one<64, false, 2>();
    if (e != cudaSuccess || !kv8) return e;
    e = head_dim == 128 ? configure_one<128, true, 2>() : configure_one<64, true, 2>();
    if (e != cudaSuccess) return e;
    return head_dim == 128 ? configure_one<128, true, 1>() : configure_one<64, true, 1>();
}

// kv8: the pool tensor maps are over E4M3 codes; one_q_tile: the plan has no pair-mode unit
cudaError_t launch_fwd(const FwdParams &p, int head_dim, bool kv8, bool one_q_tile, int num_ctas, cudaStream_t stream)
{
    if (num_ctas <= 0) return cudaSuccess;
    if (head_dim == 128) {
        if (!kv8) launch_one<128, false, 2>(p, num_ctas, stream);
        else if (one_q_tile) launch_one<128, true, 1>(p, num_ctas, stream);
        else launch_one<128, true, 2>(p, num_ctas, stream);
    } else {
        if (!kv8) launch_one<64, false, 2>(p, num_ctas, stream);
        else if (one_q_tile) launch_one<64, true, 1>(p, num_ctas, stream);
        else launch_one<64, true, 2>(p, num_ctas, stream);
    }
    return cudaGetLastError();
}

}  // namespace msa

#ifdef MSA_PROF
// profiling builds only (never the shipped library): copy out and clear the role counters
extern "C" int msa_debug_read_prof(unsigned long long *host)
{
    cudaError_t e = cudaMemcpyFromSymbol(host, msa::g_prof, sizeof(msa::g_prof));
    if (e != cudaSuccess) return -1;
    static unsigned long long zero[160][32];
    e = cudaMemcpyToSymbol(msa::g_prof, zero, sizeof(zero));
    return e == cudaSuccess ? 0 : -1;
}
extern "C" int msa_debug_read_trace(long long *host)
{
    return cudaMemcpyFromSymbol(host, msa::g_trace, sizeof(msa::g_trace)) == cudaSuccess ? 0 : -1;
}
#endif
