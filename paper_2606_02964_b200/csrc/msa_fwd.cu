// Forward-kernel launcher for libmsa (sm_100a only).
#include "msa_fwd_pipe.cuh"

namespace msa {

template <int D, bool KV8>
static cudaError_t configure_one()
{
    return cudaFuncSetAttribute(msa_fwd_pipe_kernel<D, KV8>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                PipeCfg<D, KV8>::kSmemBytes);
}

template <int D, bool KV8>
static void launch_one(const FwdParams &p, int num_ctas, cudaStream_t stream)
{
    msa_fwd_pipe_kernel<D, KV8><<<num_ctas, 512, PipeCfg<D, KV8>::kSmemBytes, stream>>>(p);
}

// The kernel needs more dynamic shared memory than the default limit; the attribute is per device and
// per function, so the handle sets it once for its own device (msa_create).  kv8: the fp8-pool variant.
cudaError_t configure_fwd(int head_dim, bool kv8)
{
    if (head_dim == 128) return kv8 ? configure_one<128, true>() : configure_one<128, false>();
    return kv8 ? configure_one<64, true>() : configure_one<64, false>();
}

cudaError_t launch_fwd(const FwdParams &p, int head_dim, bool kv8, int num_ctas, cudaStream_t stream)
{
    if (num_ctas <= 0) return cudaSuccess;
    if (head_dim == 128) {
        if (kv8) launch_one<128, true>(p, num_ctas, stream);
        else launch_one<128, false>(p, num_ctas, stream);
    } else {
        if (kv8) launch_one<64, true>(p, num_ctas, stream);
        else launch_one<64, false>(p, num_ctas, stream);
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
