// epi_math.cuh -- epilogue arithmetic shared by the tcgen05 GEMM (tc_gemm.cu) and the fused post-attention block
// (tc_post.cu): the activation of reading A5/A6 on packed fp32 pairs, bf16 hi + lo splitting.
#pragma once
#include "common.cuh"
#include "ptx.cuh"

namespace mlpf {

// exact-erf GELU (reading A6) on two values, erf from Abramowitz & Stegun 7.1.26 (|error| <= 1.5e-7):
//   GELU(x) = x/2 + |x| (1/2 - p(t) e^{-x^2/2} / 2),  t = 1 / (1 + 0.3275911 |x| / sqrt 2)
// (= max(x, 0) - |x| p e / 2: for x < 0 this is 0.5 x (1 - erf|x/sqrt 2|); the two halves x/2 and |x|/2 cancel exactly
// up to the rounding of the last FMA).  The factor -1/2 is folded into the polynomial's coefficients.  4 MUFU + 13 other
// issue slots per PAIR (packed FFMA2 / FMUL2; |x| is two LOP3) instead of erff's ~40 per value: the activation epilogues
// are issue-bound.
__device__ __forceinline__ float2 gelu2(float2 x) {
    const float2 ax = make_float2(fabsf(x.x), fabsf(x.y));
    const float2 d = ptx::ffma2(ax, make_float2(0.23164189f, 0.23164189f), make_float2(1.0f, 1.0f));
    float2 t;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(t.x) : "f"(d.x));
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(t.y) : "f"(d.y));
    float2 p = ptx::ffma2(t, make_float2(-0.5f * 1.061405429f, -0.5f * 1.061405429f), make_float2(0.5f * 1.453152027f, 0.5f * 1.453152027f));
    p = ptx::ffma2(p, t, make_float2(-0.5f * 1.421413741f, -0.5f * 1.421413741f));
    p = ptx::ffma2(p, t, make_float2(0.5f * 0.284496736f, 0.5f * 0.284496736f));
    p = ptx::ffma2(p, t, make_float2(-0.5f * 0.254829592f, -0.5f * 0.254829592f));
    p = ptx::fmul2(p, t);                                                                                        // -p(t) / 2
    const float2 xx = ptx::fmul2(ptx::fmul2(x, x), make_float2(-0.72134752044448170f, -0.72134752044448170f));  // -x^2/2 log2 e
    const float2 e = make_float2(ptx::fast_exp2(xx.x), ptx::fast_exp2(xx.y));
    const float2 w = ptx::ffma2(p, e, make_float2(0.5f, 0.5f));                                                  // 1/2 - p e / 2
    return ptx::ffma2(ax, w, ptx::fmul2(x, make_float2(0.5f, 0.5f)));
}

template <int ACT>
__device__ __forceinline__ float2 act2(float2 v) {
    if (ACT == ACT_GELU) return gelu2(v);
    if (ACT == ACT_RELU) return make_float2(fmaxf(v.x, 0.0f), fmaxf(v.y, 0.0f));
    return v;
}

// v -> bf16 pair hi = T(v) and lo = T(v - hi): bf16 -> fp32 is a 16-bit shift
__device__ __forceinline__ void split_bf16x2(float2 v, uint32_t& hi, uint32_t& lo) {
    __nv_bfloat162 h2 = __floats2bfloat162_rn(v.x, v.y);
    hi = *reinterpret_cast<uint32_t*>(&h2);
    const float2 d = ptx::fadd2(v, make_float2(-__uint_as_float(hi << 16), -__uint_as_float(hi & 0xffff0000u)));
    __nv_bfloat162 l2 = __floats2bfloat162_rn(d.x, d.y);
    lo = *reinterpret_cast<uint32_t*>(&l2);
}

}  // namespace mlpf
