// Forward-kernel launchers for libmsa (sm_100a only).
#include "msa_fwd_pipe.cuh"
#include "msa_fwd_simple.cuh"

namespace msa {

int fwd_tiles_per_group(FwdVariant v)
{
    return v == FwdVariant::Simple ? 1 : 2;
}

template <int D>
static cudaError_t launch_simple(const FwdParams &p, int num_ctas, cudaStream_t stream)
{
    using C = SimpleCfg<D>;
    static bool configured = false;
    if (!configured) {
        cudaError_t e = cudaFuncSetAttribute(msa_fwd_simple_kernel<D>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                             C::kSmemBytes);
        if (e != cudaSuccess) return e;
        configured = true;
    }
    msa_fwd_simple_kernel<D><<<num_ctas, 128, C::kSmemBytes, stream>>>(p);
    return cudaGetLastError();
}

template <int D>
static cudaError_t launch_pipe(const FwdParams &p, int num_ctas, cudaStream_t stream)
{
    using C = PipeCfg<D>;
    static bool configured = false;
    if (!configured) {
        cudaError_t e = cudaFuncSetAttribute(msa_fwd_pipe_kernel<D>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                             C::kSmemBytes);
        if (e != cudaSuccess) return e;
        configured = true;
    }
    msa_fwd_pipe_kernel<D><<<num_ctas, 512, C::kSmemBytes, stream>>>(p);
    return cudaGetLastError();
}

cudaError_t launch_fwd(const FwdParams &p, int head_dim, int num_ctas, FwdVariant v, cudaStream_t stream)
{
    if (num_ctas <= 0) return cudaSuccess;
    if (v == FwdVariant::Simple)
        return head_dim == 128 ? launch_simple<128>(p, num_ctas, stream) : launch_simple<64>(p, num_ctas, stream);
    return head_dim == 128 ? launch_pipe<128>(p, num_ctas, stream) : launch_pipe<64>(p, num_ctas, stream);
}

}  // namespace msa
