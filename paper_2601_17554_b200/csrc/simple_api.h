// simple_api.h -- host-side launchers of the CUDA-core kernels (simple_kernels.cu).  `fp32` selects the
// element type of activations / weights (float for the fp32 debug path, bf16 otherwise).
#pragma once
#include "common.cuh"

namespace mlpf {

constexpr int SCHED_BLOCK = 1024;
constexpr int EMB_ROWS = 64;
constexpr int MAX_OUT = 24;
constexpr int MAX_HBLK = 6;        // head blocks: [binary] + PID + up to 4 regression heads (L156: "six two-layer FFN heads")
struct HeadsOut {
    int n_out; int n_bin; int n_cls; int n_reg;     // outputs in this order: binary (0 | 1), class logits, regressions
    int blk[MAX_OUT];
};

// pad-row compaction arrays of a0 (oracle.schedule: comp_row, offsets_c, comp_type_perm), all device pointers
struct SchedCompact {
    int *block_vbase, *n_comp;        // [blocks], [1]: valid rows before each 1024-row block, total valid rows
    int *vbefore, *comp_row;          // [N]
    int *orig_row, *row_event_c;      // [N] indexed by compacted row
    int *comp_type_perm;              // [type_offsets[5]]: sorted slot -> compacted row
    int *offsets_c;                   // [E + 1]
};
// a0 device half: 4 launches.  Returns the number of kernels launched.
int launch_schedule(const float* X, int N, int F, const int* offsets, int E, int* block_counts, int* block_base,
                    int* valid, uint32_t* valid_bits, int* row_event, int* row_pos, int* n_valid, int* type_offsets, int* sorted_row,
                    int* type_perm, const SchedCompact& sc, cudaStream_t st);
void launch_uncompact(const float* src, const int* comp_row, float* out, int64_t N, int cols, cudaStream_t st);
// X [N, F <= 64] fp32 -> xa [slots, 192] bf16 = [x_hi | x_lo | x_hi] at the rows' type-sorted slots (pad rows skipped)
void launch_embed_pack(const float* X, int N, int F, const int* sorted_row, void* xa, cudaStream_t st);
void launch_embed_l1(bool fp32, const float* X, int N, int F, int d, const float* W1t, const float* b1, int act,
                     const int* sorted_row, void* h1, void* h1_lo, float* h, cudaStream_t st);
int launch_layernorm(bool fp32, int d, const float* x, int N, const float* g, const float* b, float eps, void* u,
                     void* u_lo, cudaStream_t st, uint8_t* u8 = nullptr, float u8_scale = 1.0f);
void launch_gemm_simple(bool fp32, const void* A, const void* A_lo, const void* W, int M, int N, int K, const Epi& ep,
                        cudaStream_t st);
void launch_attn_simple(bool fp32, int hd, const void* QKV, const int* key_valid,
                        const int* offsets, const int2* work, int n_tiles, int H, int tile_q, int d, void* O,
                        void* O_lo, cudaStream_t st);
void launch_heads_l2(bool fp32, const void* hidden, const void* hidden_lo, int N, int d, int ld_hidden,
                     const float* W2, const float* b2, const int* valid, const int* hid_row, const HeadsOut& ho, float* out_logits,
                     float* out_regress, float* out_binary, cudaStream_t st);
void launch_sched_replicate(int N, int N_pad, int E, int g, int d, int* offsets, int* n_valid, int* row_event, int* valid,
                            uint32_t* valid_bits, float* h, cudaStream_t st);
// bits[i / 32] bit (i % 32) = valid[i] != 0; `bits` holds (N + 31) / 32 words (+ 3 zero words for the attention kernel)
void launch_pack_valid_bits(const int* valid, int N, uint32_t* bits, cudaStream_t st);
void launch_cast_rows(bool fp32, const float* h, int64_t n, void* u, void* u_lo, cudaStream_t st);
void launch_untile_h(const float* h_tiled, float* out, int64_t N, int d, cudaStream_t st);
float launch_microbench(int which, int iters, int num_sms, cudaStream_t st);
void launch_to_f32(bool fp32, const void* src, float* dst, int64_t n, cudaStream_t st);

}  // namespace mlpf
