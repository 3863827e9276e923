// common.cuh -- shared device-side types of libmlpf.so (sm_100a only).
#pragma once
#include <cuda_runtime.h>
#include <cuda_bf16.h>
#include <stdint.h>
#include <cstdio>

namespace mlpf {

typedef __nv_bfloat16 bf16;

enum Act { ACT_NONE = 0, ACT_RELU = 1, ACT_GELU = 2 };

// activation between the two linears of every 2-layer FFN (reading A5/A6)
__device__ __forceinline__ float apply_act(float x, int act) {
    if (act == ACT_RELU) return fmaxf(x, 0.0f);
    if (act == ACT_GELU) return 0.5f * x * (1.0f + erff(x * 0.70710678118654752440f));
    return x;
}

template <typename T> __device__ __forceinline__ float to_f32(T v);
template <> __device__ __forceinline__ float to_f32<float>(float v) { return v; }
template <> __device__ __forceinline__ float to_f32<bf16>(bf16 v) { return __bfloat162float(v); }
template <typename T> __device__ __forceinline__ T from_f32(float v);
template <> __device__ __forceinline__ float from_f32<float>(float v) { return v; }
template <> __device__ __forceinline__ bf16 from_f32<bf16>(float v) { return __float2bfloat16_rn(v); }

// Epilogue description shared by the CUDA-core GEMM and the tcgen05 GEMM:
//   v = acc + bias[n]; v = act(v); v += residual[m, n];
//   out_f32[row, n] = v;  out_act[row, n] = T(v) (+ out_act_lo[row, n] = T(v - T(v)))
// row = row_perm ? row_perm[m] : m (row < 0: nothing is written).  Grouped mode (group_offsets != null):
// the M-tile starting at m0 uses weight/bias block g-1 where group_offsets[g] <= m0 < group_offsets[g+1]
// (g = 1..n_groups, segments are multiples of 128 rows); tiles at or beyond group_offsets[n_groups+1] exit.
struct Epi {
    const float* bias = nullptr;
    int act = ACT_NONE;
    const float* residual = nullptr; int64_t ld_res = 0;
    float* out_f32 = nullptr;        int64_t ld_f32 = 0;
    void* out_act = nullptr;         int64_t ld_act = 0;
    void* out_act_lo = nullptr;      // optional second bf16 term: out_act_lo = T(v - out_act), same ld
    const int* row_perm = nullptr;
    const int* group_offsets = nullptr;
    int n_groups = 0;
    // Uniform groups (two parallel encoders): group_rows > 0 (a multiple of 128) -> the M-tile starting at
    // m0 uses weight / bias block m0 / group_rows of a weight matrix [G * N, K] and a bias [G * N].
    int group_rows = 0;
    // Pad-row compaction: nc_dev (device, may be null) holds the number of meaningful rows (per group when group_rows > 0);
    // M-tiles that start at or beyond it are skipped (the host only knows the upper bound M).
    const int* nc_dev = nullptr;
    // FP8 operands (NEXT-3): the accumulator is multiplied by out_scale = 1 / (scale_A scale_W) before the bias
    float out_scale = 1.0f;
    // QKV projection only (a3 -> a4): the epilogue also emits the attention kernel's softmax bound inputs (tc_attn2.cu):
    // qn[row, head] = |q_row| per head and kmax[event, head] = max |k_row| (atomicMax on the float bits; zeroed by the
    // caller), from the fp32 values before the bf16 rounding (the consumer pads the bound by 2^-7).  Columns [0, nd) are
    // q, [nd, 2 nd) k; heads are nhd columns wide; row_event gives the (compacted) row's event.
    float* qn = nullptr; float* kmax = nullptr; const int* row_event = nullptr;
    int nH = 0, nhd = 0, nd = 0;
    // with qn set: columns [0, nd) (q) are multiplied by q_scale (= log2(e) / sqrt(hd), the softmax scale) before the bf16
    // rounding, and qn is the norm of the scaled values: the attention kernel then exponentiates S = q k as it is
    float q_scale = 1.0f;
};

__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
__device__ __forceinline__ float warp_max(float v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, o));
    return v;
}

}  // namespace mlpf
