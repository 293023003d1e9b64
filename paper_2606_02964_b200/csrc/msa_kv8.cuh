// fp8 (E4M3) pool: the exact code -> bf16 conversion shared by the forward kernel's converter warps (msa_fwd_pipe.cuh)
// and the dequantising pre-pass (msa_dequant.cu).
#pragma once
#include <stdint.h>

namespace msa {

// ---------------------------------------------------------------- KV8: E4M3 codes -> bf16, exactly
// Two codes -> two bf16 = code * 2^k.  cvt gives the exact f16 pair (one ALU-pipe instruction); each half is widened
// to f32 and multiplied by the KV head's scale in one mixed-precision FMA (fma.rn.f32.f16: f16 inputs, f32 result,
// exact -- the product has four significant bits); the bf16 pair is the two high halves of those f32 (PRMT: nothing
// is rounded).  Two ALU-pipe and two FMA-pipe instructions per pair; shifting the f16 fields into place and rebiasing
// with a bf16 multiply instead costs four ALU-pipe instructions and measured 1.5x slower (profiles/r02_microbench.md).
// `mul` = f16 bits of 2^k in the low half.
__device__ __forceinline__ uint32_t e4m3x2_to_bf16x2(uint32_t two_codes, uint32_t mul)
{
    uint32_t h, r;
    float lo, hi;
    asm("cvt.rn.f16x2.e4m3x2 %0, %1;" : "=r"(h) : "h"(static_cast<uint16_t>(two_codes)));
    asm("{\n\t.reg .b16 a, b;\n\tmov.b32 {a, b}, %2;\n\tfma.rn.f32.f16 %0, a, %3, 0f00000000;\n\tfma.rn.f32.f16 %1, b, %3, 0f00000000;\n\t}"
        : "=f"(lo), "=f"(hi) : "r"(h), "h"(static_cast<uint16_t>(mul)));
    asm("prmt.b32 %0, %1, %2, 0x7632;" : "=r"(r) : "r"(__float_as_uint(lo)), "r"(__float_as_uint(hi)));
    return r;
}

// Two codes -> code * 2^k as an f16 pair, exactly (the short-query variant multiplies in f16): cvt gives the codes' exact f16
// image, one packed multiply applies the KV head's scale.  For every legal k in [-14, 7] the product is an f16 -- the
// largest, 448 * 2^7 = 57344, is below 65504 and the smallest, the subnormal code 2^-9 times 2^-14 = 2^-23, is a multiple of
// f16's 2^-24 -- so nothing is rounded.  `mul2` = f16 bits of 2^k in both halves.
__device__ __forceinline__ uint32_t e4m3x2_to_f16x2(uint32_t two_codes, uint32_t mul2)
{
    uint32_t h, r;
    asm("cvt.rn.f16x2.e4m3x2 %0, %1;" : "=r"(h) : "h"(static_cast<uint16_t>(two_codes)));
    asm("mul.rn.f16x2 %0, %1, %2;" : "=r"(r) : "r"(h), "r"(mul2));
    return r;
}

}  // namespace msa
