// Forward-kernel launcher for libmsa (sm_100a only).
#include "msa_fwd_pipe.cuh"

namespace msa {

int fwd_smem_bytes(int head_dim)
{
    return head_dim == 128 ? PipeCfg<128>::kSmemBytes : PipeCfg<64>::kSmemBytes;
}

// The kernel needs more dynamic shared memory than the default limit; the attribute is per device and
// per function, so the handle sets it once for its own device (msa_create).
cudaError_t configure_fwd(int head_dim)
{
    if (head_dim == 128)
        return cudaFuncSetAttribute(msa_fwd_pipe_kernel<128>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                    PipeCfg<128>::kSmemBytes);
    return cudaFuncSetAttribute(msa_fwd_pipe_kernel<64>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                PipeCfg<64>::kSmemBytes);
}

cudaError_t launch_fwd(const FwdParams &p, int head_dim, int num_ctas, cudaStream_t stream)
{
    if (num_ctas <= 0) return cudaSuccess;
    if (head_dim == 128)
        msa_fwd_pipe_kernel<128><<<num_ctas, 512, PipeCfg<128>::kSmemBytes, stream>>>(p);
    else
        msa_fwd_pipe_kernel<64><<<num_ctas, 512, PipeCfg<64>::kSmemBytes, stream>>>(p);
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
