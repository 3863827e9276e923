// tc_gemm.cuh -- tcgen05 / TMEM / TMA GEMM for sm_100a:  C[M,N] = A[M,K] W[N,K]^T  (+ shared epilogue).
// Steps a1 (second layer), a3, a5, a6, a7, a8 (first layer) of DESIGN.md; contractions of PAPER.md L148-L156.
//
// One CTA computes a 128 x BLOCK_N tile.  Warp 0 = TMA producer (128B-swizzled K-major tiles of 64 bf16
// columns into a ring of shared-memory stages), warp 1 = MMA issuer (one elected thread, tcgen05.mma
// kind::f16, fp32 accumulator in TMEM), warps 2..5 = epilogue (tcgen05.ld, one accumulator row per thread).
// Two CTAs are co-resident per SM so one tile's epilogue overlaps the other's main loop.
// SPLIT: A is given as two bf16 terms (A = A_hi + A_lo); both are multiplied by the same W tile into the
// same accumulator, so activation rounding is ~2^-17 instead of 2^-9.
#include "tc_api.h"
#include "ptx.cuh"

namespace mlpf {

int tc_init(TcContext* c) {
    c->err[0] = 0;
    void* fn = nullptr;
    cudaDriverEntryPointQueryResult q;
    cudaError_t e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &q);
    if (e != cudaSuccess || q != cudaDriverEntryPointSuccess || !fn) {
        snprintf(c->err, sizeof c->err, "cuTensorMapEncodeTiled not available (%s)", cudaGetErrorString(e));
        return -1;
    }
    c->encode = (PFN_encodeTiled)fn;
    int dev = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&c->num_sms, cudaDevAttrMultiProcessorCount, dev);
    return 0;
}

int tc_tensor_map(TcContext* c, CUtensorMap* out, const void* ptr, uint64_t d0, uint64_t d1, uint64_t ld,
                         uint32_t b0, uint32_t b1) {
    const uint32_t sw_bytes = b0 * 2;
    TcContext::Key key{ptr, d0, d1, ld, b0, b1, sw_bytes};
    std::lock_guard<std::mutex> lk(c->mu);
    auto it = c->cache.find(key);
    if (it != c->cache.end()) { *out = it->second; return 0; }
    CUtensorMapSwizzle sw = sw_bytes == 128 ? CU_TENSOR_MAP_SWIZZLE_128B
                          : sw_bytes == 64  ? CU_TENSOR_MAP_SWIZZLE_64B
                          : sw_bytes == 32  ? CU_TENSOR_MAP_SWIZZLE_32B : CU_TENSOR_MAP_SWIZZLE_NONE;
    cuuint64_t dims[2] = {d0, d1};
    cuuint64_t strides[1] = {ld * 2};
    cuuint32_t box[2] = {b0, b1};
    cuuint32_t estr[2] = {1, 1};
    alignas(64) CUtensorMap tm;
    CUresult r = c->encode(&tm, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<void*>(ptr), dims, strides, box, estr,
                           CU_TENSOR_MAP_INTERLEAVE_NONE, sw, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                           CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) {
        snprintf(c->err, sizeof c->err, "cuTensorMapEncodeTiled failed (%d) ptr=%p dims=(%llu,%llu) ld=%llu box=(%u,%u)",
                 (int)r, ptr, (unsigned long long)d0, (unsigned long long)d1, (unsigned long long)ld, b0, b1);
        return -1;
    }
    if (c->cache.size() > 4096) c->cache.clear();
    c->cache.emplace(key, tm);
    *out = tm;
    return 0;
}

// ------------------------------------------------------------------------------------------------ kernel
constexpr int GEMM_BM = 128, GEMM_BK = 64;
constexpr int GEMM_THREADS = 192;

template <int BLOCK_N, int STAGES, bool SPLIT>
struct GemmCfg {
    static constexpr int A_BYTES = GEMM_BM * GEMM_BK * 2;            // 16 KB per A term
    static constexpr int B_BYTES = BLOCK_N * GEMM_BK * 2;
    static constexpr int STAGE_BYTES = A_BYTES * (SPLIT ? 2 : 1) + B_BYTES;
    static constexpr int SMEM_BYTES = STAGES * STAGE_BYTES + 1024;   // + slack for 1024 B alignment
    static constexpr int TMEM_COLS = BLOCK_N < 32 ? 32 : BLOCK_N;
};

// epilogue of one 32-column chunk held in registers (thread = one row)
template <typename = void>
__device__ __forceinline__ void gemm_epilogue_chunk(const uint32_t (&acc)[32], const Epi& ep, int64_t w_row0, int row,
                                                    int n_base, bool row_ok) {
    float v[32];
#pragma unroll
    for (int j = 0; j < 32; ++j) {
        float x = __uint_as_float(acc[j]);
        if (ep.bias) x += __ldg(ep.bias + w_row0 + n_base + j);
        v[j] = apply_act(x, ep.act);
    }
    if (!row_ok) return;
    if (ep.residual) {
        const float4* rp = reinterpret_cast<const float4*>(ep.residual + (int64_t)row * ep.ld_res + n_base);
#pragma unroll
        for (int j = 0; j < 8; ++j) {
            float4 r = rp[j];
            v[4 * j] += r.x; v[4 * j + 1] += r.y; v[4 * j + 2] += r.z; v[4 * j + 3] += r.w;
        }
    }
    if (ep.out_f32) {
        float4* op = reinterpret_cast<float4*>(ep.out_f32 + (int64_t)row * ep.ld_f32 + n_base);
#pragma unroll
        for (int j = 0; j < 8; ++j) op[j] = make_float4(v[4 * j], v[4 * j + 1], v[4 * j + 2], v[4 * j + 3]);
    }
    if (ep.out_act) {
        uint32_t hi[16], lo[16];
#pragma unroll
        for (int j = 0; j < 16; ++j) {
            __nv_bfloat162 h2 = __floats2bfloat162_rn(v[2 * j], v[2 * j + 1]);
            hi[j] = *reinterpret_cast<uint32_t*>(&h2);
            if (ep.out_act_lo) {
                __nv_bfloat162 l2 = __floats2bfloat162_rn(v[2 * j] - __low2float(h2), v[2 * j + 1] - __high2float(h2));
                lo[j] = *reinterpret_cast<uint32_t*>(&l2);
            }
        }
        uint4* op = reinterpret_cast<uint4*>((bf16*)ep.out_act + (int64_t)row * ep.ld_act + n_base);
#pragma unroll
        for (int j = 0; j < 4; ++j) op[j] = make_uint4(hi[4 * j], hi[4 * j + 1], hi[4 * j + 2], hi[4 * j + 3]);
        if (ep.out_act_lo) {
            uint4* lp = reinterpret_cast<uint4*>((bf16*)ep.out_act_lo + (int64_t)row * ep.ld_act + n_base);
#pragma unroll
            for (int j = 0; j < 4; ++j) lp[j] = make_uint4(lo[4 * j], lo[4 * j + 1], lo[4 * j + 2], lo[4 * j + 3]);
        }
    }
}

template <int BLOCK_N, int STAGES, bool SPLIT>
__global__ void __launch_bounds__(GEMM_THREADS)
k_tc_gemm(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmA_lo,
          const __grid_constant__ CUtensorMap tmB, int M, int N, int K, Epi ep) {
    using Cfg = GemmCfg<BLOCK_N, STAGES, SPLIT>;
    extern __shared__ uint8_t smem_raw[];
    __shared__ uint64_t bars[2 * STAGES + 1];
    __shared__ uint32_t tmem_base_slot;

    const int warp = ptx::uniform_warp_idx(), lane = threadIdx.x & 31;
    const int m0 = blockIdx.y * GEMM_BM, n0 = blockIdx.x * BLOCK_N;
    int64_t w_row0 = 0;
    if (ep.group_offsets) {                                   // grouped GEMM (per-type embedding weights)
        if (m0 >= ep.group_offsets[ep.n_groups + 1]) return;  // CTA-uniform, before any barrier / allocation
        int g = 1;
        while (g < ep.n_groups && m0 >= ep.group_offsets[g + 1]) ++g;
        w_row0 = (int64_t)(g - 1) * N;
    }
    const uint32_t smem_base = (ptx::smem_u32(smem_raw) + 1023u) & ~1023u;
    const uint32_t bar_full = ptx::smem_u32(&bars[0]);
    const uint32_t bar_empty = ptx::smem_u32(&bars[STAGES]);
    const uint32_t bar_acc = ptx::smem_u32(&bars[2 * STAGES]);

    if (warp == 0 && lane == 0) {
        for (int s = 0; s < STAGES; ++s) { ptx::mbar_init(bar_full + 8 * s, 1); ptx::mbar_init(bar_empty + 8 * s, 1); }
        ptx::mbar_init(bar_acc, 1);
        ptx::fence_barrier_init();
        ptx::tma_prefetch_desc(&tmA);
        ptx::tma_prefetch_desc(&tmB);
        if (SPLIT) ptx::tma_prefetch_desc(&tmA_lo);
    }
    if (warp == 1) {
        ptx::tmem_alloc(ptx::smem_u32(&tmem_base_slot), Cfg::TMEM_COLS);
        ptx::tmem_relinquish();
    }
    ptx::tc_fence_before();
    __syncthreads();
    ptx::tc_fence_after();
    const uint32_t tmem_base = tmem_base_slot;
    const int num_kb = K / GEMM_BK;

    if (warp == 0) {
        // ---------------- TMA producer
        for (int kb = 0; kb < num_kb; ++kb) {
            const int s = kb % STAGES;
            const uint32_t ph = (kb / STAGES) & 1;
            ptx::mbar_wait(bar_empty + 8 * s, ph ^ 1);
            if (lane == 0) {
                const uint32_t st = smem_base + s * Cfg::STAGE_BYTES;
                ptx::mbar_expect_tx(bar_full + 8 * s, Cfg::STAGE_BYTES);
                ptx::tma_load_2d(st, &tmA, bar_full + 8 * s, kb * GEMM_BK, m0);
                if (SPLIT) ptx::tma_load_2d(st + Cfg::A_BYTES, &tmA_lo, bar_full + 8 * s, kb * GEMM_BK, m0);
                ptx::tma_load_2d(st + Cfg::A_BYTES * (SPLIT ? 2 : 1), &tmB, bar_full + 8 * s, kb * GEMM_BK, (int)(w_row0 + n0));
            }
            __syncwarp();
        }
    } else if (warp == 1) {
        // ---------------- MMA issuer
        constexpr uint32_t idesc = ptx::umma_idesc_bf16(GEMM_BM, BLOCK_N);
        for (int kb = 0; kb < num_kb; ++kb) {
            const int s = kb % STAGES;
            const uint32_t ph = (kb / STAGES) & 1;
            ptx::mbar_wait(bar_full + 8 * s, ph);
            ptx::tc_fence_after();
            {   // all lanes, warp-uniform operands: one lane is elected inside the MMA / commit wrappers
                const uint32_t a_addr = smem_base + s * Cfg::STAGE_BYTES;
                const uint32_t b_addr = a_addr + Cfg::A_BYTES * (SPLIT ? 2 : 1);
#pragma unroll
                for (int k = 0; k < GEMM_BK / 16; ++k) {
                    const uint64_t bd = ptx::umma_desc_kmajor(b_addr + k * 32, 128);
                    ptx::mma_ss(tmem_base, ptx::umma_desc_kmajor(a_addr + k * 32, 128), bd, idesc, (kb | k) != 0);
                    if (SPLIT) ptx::mma_ss(tmem_base, ptx::umma_desc_kmajor(a_addr + Cfg::A_BYTES + k * 32, 128), bd, idesc, 1);
                }
                ptx::mma_commit(bar_empty + 8 * s);           // frees the stage when these MMAs retire
                if (kb == num_kb - 1) ptx::mma_commit(bar_acc);
            }
        }
    } else {
        // ---------------- epilogue: warp w reads TMEM lanes 32*(w%4) .. +31
        const int q = warp & 3;
        const int m = m0 + q * 32 + lane;
        const bool row_ok = m < M;
        int row = m;
        if (row_ok && ep.row_perm) row = ep.row_perm[m];
        const bool write_ok = row_ok && row >= 0;
        ptx::mbar_wait(bar_acc, 0);
        ptx::tc_fence_after();
#pragma unroll 1
        for (int c = 0; c < BLOCK_N; c += 32) {
            uint32_t acc[32];
            ptx::tmem_ld32(tmem_base + ((uint32_t)(q * 32) << 16) + c, acc);
            ptx::tmem_ld_wait();
            gemm_epilogue_chunk(acc, ep, w_row0, row, n0 + c, write_ok);
        }
    }
    ptx::tc_fence_before();
    __syncthreads();
    if (warp == 1) ptx::tmem_dealloc(tmem_base, Cfg::TMEM_COLS);
}

// ------------------------------------------------------------------------------------------------ launch
template <int BLOCK_N, int STAGES, bool SPLIT>
static int tc_gemm_launch_cfg(TcContext* c, const bf16* A, const bf16* A_lo, const bf16* W, int M, int N, int K,
                              int w_rows, const Epi& ep, cudaStream_t st) {
    using Cfg = GemmCfg<BLOCK_N, STAGES, SPLIT>;
    CUtensorMap tmA, tmAlo, tmB;
    if (tc_tensor_map(c, &tmA, A, K, M, K, GEMM_BK, GEMM_BM)) return -1;
    if (SPLIT) { if (tc_tensor_map(c, &tmAlo, A_lo, K, M, K, GEMM_BK, GEMM_BM)) return -1; }
    else tmAlo = tmA;
    if (tc_tensor_map(c, &tmB, W, K, w_rows, K, GEMM_BK, BLOCK_N)) return -1;
    auto kern = k_tc_gemm<BLOCK_N, STAGES, SPLIT>;
    static bool attr_set = false;
    if (!attr_set) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, Cfg::SMEM_BYTES);
        if (e != cudaSuccess) { snprintf(c->err, sizeof c->err, "cudaFuncSetAttribute: %s", cudaGetErrorString(e)); return -1; }
        attr_set = true;
    }
    dim3 grid(N / BLOCK_N, (M + GEMM_BM - 1) / GEMM_BM);
    kern<<<grid, GEMM_THREADS, Cfg::SMEM_BYTES, st>>>(tmA, tmAlo, tmB, M, N, K, ep);
    return 0;
}

int tc_gemm_launch(TcContext* c, const bf16* A, const bf16* A_lo, const bf16* W, int M, int N, int K,
                          const Epi& ep, cudaStream_t st) {
    if (N % 64 || K % 64) { snprintf(c->err, sizeof c->err, "tc_gemm: N=%d, K=%d must be multiples of 64", N, K); return -1; }
    const int w_rows = ep.group_offsets ? ep.n_groups * N : N;
    if (N % 128 == 0) {
        return A_lo ? tc_gemm_launch_cfg<128, 2, true>(c, A, A_lo, W, M, N, K, w_rows, ep, st)
                    : tc_gemm_launch_cfg<128, 3, false>(c, A, nullptr, W, M, N, K, w_rows, ep, st);
    }
    return A_lo ? tc_gemm_launch_cfg<64, 4, true>(c, A, A_lo, W, M, N, K, w_rows, ep, st)
                : tc_gemm_launch_cfg<64, 4, false>(c, A, nullptr, W, M, N, K, w_rows, ep, st);
}

}  // namespace mlpf
