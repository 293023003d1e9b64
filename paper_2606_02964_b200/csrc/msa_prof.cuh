// Profiling hooks of the forward kernel (msa_fwd_pipe.cuh), kept out of the kernel source.
// Empty macros in the shipped library; a build with -DMSA_PROF (role-level cycle counters) or -DMSA_PROF=2 (event trace of
// CTA 0's first unit) is a measuring tool and never the product.
#pragma once

namespace msa {

// Optional role-level cycle counters (build with -DMSA_PROF; never in the shipped library):
// lane 0 of one warp per role accumulates clock64() deltas into g_prof[cta][slot].
#ifdef MSA_PROF
__device__ unsigned long long g_prof[160][32];
__device__ long long g_trace[4][64][12];
#define PROF_TRACE(role, step, ev) \
    do { if (blockIdx.x == 0 && u == u_begin && (step) < 64) g_trace[role][step][ev] = clock64(); } while (0)
#if MSA_PROF == 2   /* event trace only: no accumulators in the hot loops */
#define PROF_DECL()
#define PROF_T0()
#define PROF_ADD(slot)
#define PROF_INC(slot, v)
#define PROF_FLUSH(lo, hi)
#else
#define PROF_DECL() unsigned long long prof_acc[32] = {}
#define PROF_T0() const long long prof_t0_ = clock64()
#define PROF_ADD(slot) prof_acc[slot] += static_cast<unsigned long long>(clock64() - prof_t0_)
#define PROF_INC(slot, v) prof_acc[slot] += static_cast<unsigned long long>(v)
#define PROF_FLUSH(lo, hi)                                                             \
    do {                                                                               \
        _Pragma("unroll") for (int i_ = (lo); i_ < (hi); ++i_) g_prof[blockIdx.x][i_] += prof_acc[i_]; \
    } while (0)
#endif
#else
#define PROF_TRACE(role, step, ev)
#define PROF_DECL()
#define PROF_T0()
#define PROF_ADD(slot)
#define PROF_INC(slot, v)
#define PROF_FLUSH(lo, hi)
#endif

}  // namespace msa
