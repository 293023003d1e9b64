// Softmax fast path of the pipelined MSA kernel: one thread owns one packed (head, token) row
// of a 128-key score tile that sits in TMEM as fp32, and turns it into bf16 P in place
// (P aliases the first 64 columns of S).
//
// Row reference.  p = 2^(s*scale_log2 - ref) with ref an INTEGER (in log2 units).  Moving the
// reference multiplies l and O by an exact power of two, so the result does not depend on when
// the reference moves; it only has to stay close enough above/below the scores for fp32 / bf16
// range.  The fast path therefore uses the reference it was handed (stale by up to this tile),
// finds the tile's own row max alongside, and the caller moves the reference before the next
// tile.  The only hazard is overflow when a tile's scores exceed the reference by more than
// ~2^120: a guard over the WHOLE tile is evaluated before anything is stored, so the caller
// can redo the tile on the exact (max-first) path with S still intact.
//
// Pipes.  The arithmetic is spread over three pipes so that none of them alone bounds the tile
// (B200, one softmax warp per SM sub-partition; measured: MUFU.EX2 8.0 cycles per warp
// instruction, FFMA2/FADD2 2.3, F2FP 2.1):
//   * x = s*scale_log2 - ref              one FFMA2 per element pair
//   * 2^x                                  MUFU.EX2, or ex2_poly2 on the FMA/ALU pipes for EMU of
//                                          every 8 pairs
//   * row sum from the fp32 p (FADD2), row max of the raw scores (FMNMX3), bf16 pack (F2FP)
//
// Hand-off.  P is published in two halves (keys 0-63, then 64-127): `arrive_lo` is called once
// the first 32 columns of P are visible to the tensor core, so O += P V starts on the first
// half while the second half is still being exponentiated.
#pragma once
#include <math.h>

#include "msa_ptx.cuh"

namespace msa {

constexpr float kGuardLog2 = 120.f;   // largest s*scale_log2 - ref the fast path accepts

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

// One 32-column chunk: scores -> 16 packed bf16 pairs; two sum accumulators keep the
// dependent FADD2 chain short.
template <int EMU>
__device__ __forceinline__ void softmax_chunk(const uint32_t (&sr)[32], float2 sl2, float2 nr2, float2 &sa, float2 &sb,
                                              uint32_t (&pk)[16])
{
#pragma unroll
    for (int j = 0; j < 16; ++j) {
        const float2 x = ffma2(make_float2(__uint_as_float(sr[2 * j]), __uint_as_float(sr[2 * j + 1])), sl2, nr2);
        float2 pp;
        if ((j & 7) < EMU) {
            pp = ex2_poly2(x);
        } else {
            pp.x = ex2_approx(x.x);
            pp.y = ex2_approx(x.y);
        }
        if (j & 1) sb = fadd2(sb, pp); else sa = fadd2(sa, pp);
        pk[j] = pack_bf16x2(pp.x, pp.y);
    }
}

// Whole tile.  tS: TMEM address of the row's S (lane already folded in).  Returns false, with
// nothing stored, if some row of the warp failed the overflow guard.  Otherwise P is complete
// in TMEM (stores waited for, tcgen05 fence issued): `arrive_lo()` has been called for the
// first half and the caller arrives for the second.  `mark(i)` is a profiling hook (no-op in
// the shipped build).  tile_sum = sum of p against `ref`,
// tile_max = max raw score.
template <int EMU, int EMU_HI, class ArriveLo, class Mark>
__device__ __forceinline__ bool softmax_fast_tile(uint32_t tS, float sl, float ref, float &tile_sum, float &tile_max,
                                                  ArriveLo &&arrive_lo, Mark &&mark)
{
    const float2 sl2 = make_float2(sl, sl), nr2 = make_float2(-ref, -ref);
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
    softmax_chunk<EMU>(c0, sl2, nr2, sa, sb, pk0);
    // the second half has landed by now: its row max is found among the arithmetic of chunk 1,
    // so the guard is ready as soon as the first half of P is
    tmem_wait_ld_regs(c2);
    tmem_wait_ld_regs(c3);
    mx = fmaxf(mx, fmaxf(chunk_max(c2), chunk_max(c3)));
    softmax_chunk<EMU>(c1, sl2, nr2, sa, sb, pk1);
    mark(2);
    tile_max = mx;
    if (__any_sync(0xffffffffu, !(fmaf(mx, sl, -ref) <= kGuardLog2))) return false;
    mark(3);
    tmem_st16(tS, pk0);
    tmem_st16(tS + 16, pk1);
    // the first half is published one chunk later: its stores have completed by then (no stall),
    // and O += P V of keys 0-63 still finishes long before the second half is ready
    softmax_chunk<EMU_HI>(c2, sl2, nr2, sa, sb, pk0);
    tmem_wait_st();
    tc_fence_before();
    arrive_lo();
    tmem_st16(tS + 32, pk0);
    softmax_chunk<EMU_HI>(c3, sl2, nr2, sa, sb, pk1);
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
