// cand_api.h -- host-side launcher of the candidate-building kernels (candidates.cu).
#pragma once
#include "common.cuh"

namespace mlpf {

int64_t cand_scratch_bytes(int64_t N, int64_t E);
// 2 kernels + one small H2D copy on `st`; returns the launch status
cudaError_t launch_build_candidates(const float* X, int F, const int32_t* offsets_host, int E, const float* logits, int C,
                                    const float* regress, const float* binary, void* scratch, int32_t* cand_offsets, int32_t* cand_elem,
                                    int32_t* cand_pid, float* cand_p4, cudaStream_t st);

// the same with the scratch in a file-scope device array of candidates.cu (no allocation anywhere); limits below
int64_t cand_static_max_elements();
int64_t cand_static_max_events();
int64_t cand_static_bytes();
cudaError_t launch_build_candidates_static(const float* X, int F, const int32_t* offsets_host, int E, const float* logits, int C,
                                           const float* regress, const float* binary, int32_t* cand_offsets, int32_t* cand_elem,
                                           int32_t* cand_pid, float* cand_p4, cudaStream_t st);

}  // namespace mlpf
