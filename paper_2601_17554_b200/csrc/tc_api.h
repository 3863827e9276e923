// tc_api.h -- host-side interface of the tensor-core kernels (tc_gemm.cu, tc_attn.cu).
#pragma once
#include <cuda.h>
#include <mutex>
#include <unordered_map>
#include <set>
#include <utility>
#include "common.cuh"
#include "simple_api.h"

namespace mlpf {

// ------------------------------------------------------------------------------------------------ host context
typedef CUresult (*PFN_encodeTiled)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                    const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                    CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

struct TcContext {
    char err[256] = {0};
    PFN_encodeTiled encode = nullptr;
    int num_sms = 148;
    std::mutex mu;
    struct Key {
        const void* p; uint64_t d0, d1, ld; uint32_t b0, b1, sw;
        bool operator==(const Key& o) const { return p == o.p && d0 == o.d0 && d1 == o.d1 && ld == o.ld && b0 == o.b0 && b1 == o.b1 && sw == o.sw; }
    };
    struct KeyHash {
        size_t operator()(const Key& k) const {
            uint64_t h = (uint64_t)k.p * 0x9E3779B97F4A7C15ull;
            h ^= k.d0 + 0x9E3779B97F4A7C15ull + (h << 6) + (h >> 2);
            h ^= k.d1 + 0x9E3779B97F4A7C15ull + (h << 6) + (h >> 2);
            h ^= k.ld + (h << 6) + (h >> 2);
            h ^= ((uint64_t)k.b0 << 32 | k.b1) + (h << 6) + (h >> 2);
            return (size_t)(h ^ k.sw);
        }
    };
    std::unordered_map<Key, CUtensorMap, KeyHash> cache;
    std::set<std::pair<const void*, int>> attr_done;   // (kernel, device) pairs whose shared-memory limit is raised
    bool pdl = false;                                  // launch the tensor-core kernels with programmatic stream serialization
};

// kernel launch, optionally with the programmatic-stream-serialization attribute (the kernel calls ptx::grid_dep_wait())
template <typename... KArgs, typename... Args>
inline cudaError_t tc_launch(void (*kern)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, bool pdl, Args&&... args) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr; cfg.numAttrs = pdl ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, kern, std::forward<Args>(args)...);
}


int tc_init(TcContext* c);
int tc_set_smem_attr(TcContext* c, const void* kern, int bytes);
// 2D bf16 tensor map: dims (d0 inner, d1 outer), row pitch ld elements, box (b0, b1), swizzle = b0 * 2 bytes
int tc_tensor_map(TcContext* c, CUtensorMap* out, const void* ptr, uint64_t d0, uint64_t d1, uint64_t ld,
                  uint32_t b0, uint32_t b1, int elem_bytes = 2);
int tc_gemm_fp8_launch(TcContext* c, const uint8_t* A, const uint8_t* W, int M, int N, int K, const Epi& ep, cudaStream_t st);
// C = (A + A_lo) W^T with the shared epilogue; A_lo == nullptr -> plain bf16 A.  N % 64 == 0, K % 64 == 0.
int tc_gemm_launch(TcContext* c, const bf16* A, const bf16* A_lo, const bf16* W, int M, int N, int K,
                   const Epi& ep, cudaStream_t st);
// QKV [N, 3d] row-major bf16 (q | k | v).  items = (event, group) per CTA row group of tc_attn_rows_per_cta(hd)
// query rows; valid_bits: one bit per row (32 rows per word, 3 readable words past the last row's), null = all rows
// valid; n_valid [E] (valid rows per event) may be null.
int tc_attn_rows_per_cta(int hd);
int tc_attn_launch(TcContext* c, const bf16* QKV, int64_t N, const uint32_t* valid_bits, const int* n_valid,
                   const int* offsets, const int2* items, int n_items, int d, int H, bf16* O, bf16* O_lo,
                   cudaStream_t st);

// Second attention design (tc_attn2.cu): no running maximum (Cauchy-Schwarz bound from a norms pre-pass; exact two-sweep
// path for CTAs whose bound is too loose), two threads per query row.  qn [N, H], kmax [E, H]: caller-owned fp32 scratch;
// row_event [N] from the schedule.  force_exact != 0: every CTA takes the exact path (tests).  prescaled: the q columns
// of QKV (and qn) already carry the softmax scale log2(e) / sqrt(hd) (Epi::q_scale): the fast path then subtracts nothing.
int tc_attn2_rows_per_cta(int hd);
extern int g_attn2_poly_deg;         // degree of that polynomial: 3 | 2 (experiment)
extern int g_attn2_poly_every;       // tuning knob: every n-th pair of exponentials on the FMA pipe (0, 2, 3, 4; -1 = default)
int tc_attn2_launch(TcContext* c, const bf16* QKV, int64_t N, int E, const uint32_t* valid_bits, const int* n_valid,
                    const int* offsets, const int* row_event, const int2* items, int n_items, int d, int H, float* qn,
                    float* kmax, bf16* O, bf16* O_lo, int force_exact, const int* nc_dev, int group_rows, cudaStream_t st,
                    bool norms_ready = false, bool prescaled = false);

// The post-attention half of an encoder block as one kernel (tc_post.cu): h <- h + o Wo^T + bo; u2 = LN2(h);
// h <- h + act(u2 W1^T + b1) W2^T + b2; u_out = LN_next(h) (or T(h) when next_ln == 0).  d in {64, 128, 256}, dff % 128 == 0.
// n_groups > 1 (two parallel encoders): rows [g * group_rows, (g + 1) * group_rows) use weight block g of Wo [G*d, d],
// W1 [G*dff, d], W2 [G*d, dff] and vector block g (vectors are [G, len]); group_rows % 128 == 0.
struct PostArgs {
    int M = 0, d = 0, dff = 0, act = ACT_GELU, n_groups = 1, group_rows = 0;
    const int* nc_dev = nullptr;             // meaningful rows (per group) on the device: later tiles are skipped (pad-row compaction)
    const bf16 *o = nullptr, *o_lo = nullptr, *Wo = nullptr, *W1 = nullptr, *W2 = nullptr;
    const float *bo = nullptr, *ln2g = nullptr, *ln2b = nullptr, *b1 = nullptr, *b2 = nullptr, *lnng = nullptr, *lnnb = nullptr;
    float eps = 1e-5f;
    float* h = nullptr;
    int h_in_tiled = 0, h_out_tiled = 0;     // residual-stream layout in / out (tc_post.cu h_off); capacity: whole 128-row tiles
    bf16 *u_out = nullptr, *u_out_lo = nullptr;
    uint8_t* u_out_f8 = nullptr; float f8_scale = 1.0f;     // optional e4m3 copy of u_out * f8_scale
    int next_ln = 1;
    bf16 *dbg_u2 = nullptr, *dbg_g = nullptr;
};
bool tc_post_supported(int d, int dff);
int tc_post_launch(TcContext* c, const PostArgs& a, cudaStream_t st);

// All heads of step a8 as one kernel (tc_heads.cu): out = act(z W1[b]^T + b1[b]) W2[b]^T + b2[b] per head block b, hidden
// layers kept on chip.  z, z_lo [M, d] bf16 (compacted rows); W1 [n_hblk_total * d, d] bf16; W2p = the output rows packed
// per 128-column chunk as [chunk][hi | lo][16 rows][chunk columns] bf16 (tc_heads_chunk(d) columns per chunk; built by
// mlpf_create); this launch covers blocks blk0 .. blk0 + nblk - 1 (two-stack models: one launch per stack).  Outputs go to
// the ORIGINAL rows (orig_row, null = identity); the caller zeroes the output buffers first (pad rows).
struct HeadsArgs {
    int M = 0, d = 0, act = ACT_GELU, n_hblk_total = 0, blk0 = 0, nblk = 0;
    const bf16 *z = nullptr, *z_lo = nullptr, *W1 = nullptr, *W2p = nullptr;
    const float *b1 = nullptr, *b2 = nullptr;
    const int *orig_row = nullptr, *nc_dev = nullptr;
    HeadsOut ho = {};
    float *out_logits = nullptr, *out_regress = nullptr, *out_binary = nullptr;
};
bool tc_heads_supported(int d, int n_hblk);
int tc_heads_chunk(int d);
int tc_heads_launch(TcContext* c, const HeadsArgs& a, cudaStream_t st);

}  // namespace mlpf
