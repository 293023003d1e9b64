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

template <int D, int EMU, int EMU_HI>
static cudaError_t launch_pipe(const FwdParams &p, int num_ctas, cudaStream_t stream)
{
    using C = PipeCfg<D>;
    static bool configured = false;
    if (!configured) {
        cudaError_t e = cudaFuncSetAttribute(msa_fwd_pipe_kernel<D, EMU, EMU_HI>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                             C::kSmemBytes);
        if (e != cudaSuccess) return e;
        configured = true;
    }
    msa_fwd_pipe_kernel<D, EMU, EMU_HI><<<num_ctas, 512, C::kSmemBytes, stream>>>(p);
    return cudaGetLastError();
}

// emu = 10 * (pairs of 8 emulated in the first half of a tile) + (same for the second half); -1: exact path only
template <int D>
static cudaError_t launch_pipe_emu(const FwdParams &p, int num_ctas, int emu, cudaStream_t stream)
{
    switch (emu) {
    case -1: return launch_pipe<D, -1, 0>(p, num_ctas, stream);
    case 0: return launch_pipe<D, 0, 0>(p, num_ctas, stream);
    case 22: return launch_pipe<D, 2, 2>(p, num_ctas, stream);
    default: return launch_pipe<D, kDefaultEmu / 10, kDefaultEmu % 10>(p, num_ctas, stream);
    }
}

cudaError_t launch_fwd(const FwdParams &p, int head_dim, int num_ctas, FwdVariant v, int emu, cudaStream_t stream)
{
    if (num_ctas <= 0) return cudaSuccess;
    if (v == FwdVariant::Simple)
        return head_dim == 128 ? launch_simple<128>(p, num_ctas, stream) : launch_simple<64>(p, num_ctas, stream);
    return head_dim == 128 ? launch_pipe_emu<128>(p, num_ctas, emu, stream) : launch_pipe_emu<64>(p, num_ctas, emu, stream);
}

}  // namespace msa

#ifdef MSA_PROF
// profiling builds only: copy out and clear the role counters
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
