// Softmax fast path of the pipelined MSA kernel: one thread owns one packed (head, token) row
// of a 128-key score tile that sits in TMEM as fp32, and turns it into bf16 P in place
// (P aliases the first 64 columns of S).
//
// Row reference.  p = 2^(s*scale_log2 - ref) with ref an INTEGER (in log2 units).  Moving the
// reference multiplies l and O by an exact power of two, so the result does not depend on when
// the reference moves; it only has to stay close enough above/below the scores for fp32 / bf16
// range.  The fast path therefore uses the reference it was handed (stale by up to this tile),
// finds the tile's own row max alongside, and the caller moves the reference before the next
// tile.  The only hazard is overflow when a tile's scores exceed the reference by a lot: a guard
// over the WHOLE tile (score - ref <= 2^kGuardLog2) is evaluated before anything is stored, so the
// caller can redo the tile on the exact (max-first) path with S still intact.  The guard leaves
// headroom for the accumulation that follows: P <= 2^64, a tile adds at most 2^71 to l and
// 2^71 |V| to O (fp32 holds 2^127).
//
// Pipes (B200, measured with working microbenchmarks, profiles/r02_microbench.md; cycles per warp instruction on one
// SM sub-partition): MUFU.EX2 8.0; FFMA2 / FADD2 2.1; every ALU-pipe instruction (F2FP pack, FMNMX, LEA) 2.0;
// FFMA / FADD 1.0.  MUFU time overlaps with everything else, FFMA2 and ALU time add up.  An all-MUFU tile costs 1024
// cycles of MUFU per warp, about what the tensor core needs per tile and chain -- but moving part of the exponentials
// to a polynomial on the FMA / ALU pipes (measured at 4/16 ... 8/16 of the elements, with a range reduction of two
// FMAs and a degree-3 polynomial) made the kernel slower, not faster: one in-order warp per row set is bound by its
// own issue order and by the P -> PV -> QK -> S round trip, not by the MUFU pipe.
//
// Hand-off.  P is published in three steps (keys 0-63, 64-95, 96-127): `arrive(i)` is called once
// the corresponding columns of P are visible to the tensor core, so O += P V trails the
// exponentials and only the last 32 keys remain to be multiplied when the tile is done.
#pragma once
#include <math.h>

#include "msa_ptx.cuh"

namespace msa {

constexpr float kGuardLog2 = 64.f;    // largest s*scale_log2 - ref the fast path accepts (P in bf16)
constexpr float kGuardLog2F16 = 14.f; // ... when P is handed over in f16 (fp8-pool short-query variant): P <= 2^14 < 65504

struct SoftmaxRow {
    float2 sl2;       // scale_log2
    float2 nr2;       // -ref
};

__device__ __forceinline__ SoftmaxRow make_softmax_row(float sl, float ref)
{
    SoftmaxRow r;
    r.sl2 = make_float2(sl, sl);
    r.nr2 = make_float2(-ref, -ref);
    return r;
}

__device__ __forceinline__ float chunk_max(const uint32_t (&sr)[32])
{
    float a = fmaxf(__uint_as_float(sr[0]), __uint_as_float(sr[1])), b = fmaxf(__uint_as_float(sr[2]), __uint_as_float(sr[3]));
#pragma unroll
    for (int j = 4; j < 32; j += 4) {
        a = fmaxf(a, fmaxf(__uint_as_float(sr[j]), __uint_as_float(sr[j + 1])));
        b = fmaxf(b, fmaxf(__uint_as_float(sr[j + 2]), __uint_as_float(sr[j + 3])));
    }
    return fmaxf(a, b);
}

// Pairs [J0, J1) of a 32-column chunk: scores -> packed bf16 pairs; two sum accumulators keep
// the dependent FADD2 chain short.
template <int J0, int J1, bool F16 = false>
__device__ __forceinline__ void softmax_pairs(const uint32_t (&sr)[32], const SoftmaxRow &t, float2 &sa, float2 &sb,
                                              uint32_t (&pk)[16])
{
#pragma unroll
    for (int j = J0; j < J1; ++j) {
        const float s0 = __uint_as_float(sr[2 * j]), s1 = __uint_as_float(sr[2 * j + 1]);
        const float2 x = ffma2(make_float2(s0, s1), t.sl2, t.nr2);
        float2 pp;
        pp.x = ex2_approx(x.x);
        pp.y = ex2_approx(x.y);
        if (j & 1) sb = fadd2(sb, pp); else sa = fadd2(sa, pp);
        pk[j] = F16 ? pack_f16x2(pp.x, pp.y) : pack_bf16x2(pp.x, pp.y);
    }
}

// Whole tile.  tS: TMEM address of the row's S (lane already folded in).  Returns false, with
// nothing stored, if some row of the warp failed the overflow guard.  Otherwise P is complete
// in TMEM (stores waited for, tcgen05 fence issued): `arrive(0)` and `arrive(1)` have been called
// for keys 0-63 and 64-95 and the caller arrives for the rest.  `mark(i)` is a profiling hook
// (no-op in the shipped build).  tile_sum = sum of p against `ref`, tile_max = max raw score.
// The waits for the P stores name registers of the chunk computed in between (tmem_wait_st_after):
// without that the compiler is free to schedule the wait -- and the stall -- right behind the store.
template <bool F16 = false, class Arrive, class Mark>
__device__ __forceinline__ bool softmax_fast_tile(uint32_t tS, float sl, float ref, float &tile_sum,
                                                  float &tile_max, Arrive &&arrive, Mark &&mark)
{
    const SoftmaxRow t = make_softmax_row(sl, ref);
    float2 sa = make_float2(0.f, 0.f), sb = make_float2(0.f, 0.f);
    uint32_t c0[32], c1[32], c2[32], c3[32];
    uint32_t pk0[16], pk1[16];
    tmem_ld32(tS, c0);
    tmem_ld32(tS + 32, c1);
    tmem_wait_ld_regs(c0);
    tmem_wait_ld_regs(c1);
    tmem_ld32(tS + 64, c2);
    tmem_ld32(tS + 96, c3);
    mark(1);
    float mx = fmaxf(chunk_max(c0), chunk_max(c1));
    softmax_pairs<0, 16, F16>(c0, t, sa, sb, pk0);
    // the second half has landed by now: its row max is found among the arithmetic of chunk 1,
    // so the guard is ready as soon as the first half of P is
    tmem_wait_ld_regs(c2);
    tmem_wait_ld_regs(c3);
    mx = fmaxf(mx, fmaxf(chunk_max(c2), chunk_max(c3)));
    softmax_pairs<0, 16, F16>(c1, t, sa, sb, pk1);
    mark(2);
    tile_max = mx;
    if (__any_sync(0xffffffffu, !(fmaf(mx, sl, -ref) <= (F16 ? kGuardLog2F16 : kGuardLog2)))) return false;
    mark(3);
    tmem_st16(tS, pk0);
    tmem_st16(tS + 16, pk1);
    // each part is published while the next one is computed: its stores have completed by then
    // (no stall), and O += P V of the published keys finishes before the next part is ready
    softmax_pairs<0, 16, F16>(c2, t, sa, sb, pk0);
    tmem_wait_st_after(pk0[12], pk0[13], pk0[14], pk0[15]);
    tc_fence_before();
    arrive(0);
    tmem_st16(tS + 32, pk0);
    softmax_pairs<0, 8, F16>(c3, t, sa, sb, pk1);
    tmem_wait_st_after(pk1[4], pk1[5], pk1[6], pk1[7]);
    tc_fence_before();
    arrive(1);
    softmax_pairs<8, 16, F16>(c3, t, sa, sb, pk1);
    tmem_st16(tS + 48, pk1);
    tile_sum = (sa.x + sb.x) + (sa.y + sb.y);
    mark(5);
    tmem_wait_st();
    tc_fence_before();
    return true;
}

// 2^d for an integer-valued d <= 0, exactly; 0 below the normal range.
__device__ __forceinline__ float exp2_int(float d)
{
    return d < -126.f ? 0.f : __uint_as_float(static_cast<uint32_t>(static_cast<int>(d) + 127) << 23);
}

}  // namespace msa
