// tc_gemm.cu -- tcgen05 / TMEM / TMA GEMM for sm_100a:  C[M,N] = A[M,K] W[N,K]^T  (+ shared epilogue).
// Steps a1 (second layer), a3, a5, a6, a7, a8 (first layer) of DESIGN.md; contractions of PAPER.md L148-L156.
//
// Persistent kernel, one CTA per SM looping over 128 x BLOCK_N output tiles (n fastest, so the CTAs running
// at the same time share A tiles in L2).  Warp 0 = TMA producer (128B-swizzled K-major tiles of 64 bf16
// columns into a ring of shared-memory stages that runs on across tiles), warp 1 = MMA issuer (tcgen05.mma
// kind::f16, fp32 accumulators in TWO TMEM buffers), warps 2-5 and 6-9 = two epilogue warpgroups, one per
// accumulator buffer (tcgen05.ld, one accumulator row per thread): the epilogue of tile i overlaps the main
// loop of tile i+1 and the epilogue of tile i+1.
// SPLIT: A is given as two bf16 terms (A = A_hi + A_lo); both are multiplied by the same W tile into the
// same accumulator, so activation rounding is ~2^-17 instead of 2^-9.
#include "tc_api.h"
#include "ptx.cuh"
#include "epi_math.cuh"

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

// cudaFuncAttributeMaxDynamicSharedMemorySize is a per-DEVICE attribute of a kernel: set once per (kernel, device)
int tc_set_smem_attr(TcContext* c, const void* kern, int bytes) {
    int dev = 0;
    cudaGetDevice(&dev);
    {
        std::lock_guard<std::mutex> lk(c->mu);
        if (c->attr_done.count({kern, dev})) return 0;
    }
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
    if (e != cudaSuccess) { snprintf(c->err, sizeof c->err, "cudaFuncSetAttribute: %s", cudaGetErrorString(e)); return -1; }
    std::lock_guard<std::mutex> lk(c->mu);
    c->attr_done.insert({kern, dev});
    return 0;
}

int tc_tensor_map(TcContext* c, CUtensorMap* out, const void* ptr, uint64_t d0, uint64_t d1, uint64_t ld,
                         uint32_t b0, uint32_t b1, int elem_bytes) {
    const uint32_t sw_bytes = b0 * elem_bytes;
    TcContext::Key key{ptr, d0, d1, ld, b0, b1, sw_bytes + 1024u * (uint32_t)elem_bytes};
    std::lock_guard<std::mutex> lk(c->mu);
    auto it = c->cache.find(key);
    if (it != c->cache.end()) { *out = it->second; return 0; }
    CUtensorMapSwizzle sw = sw_bytes == 128 ? CU_TENSOR_MAP_SWIZZLE_128B
                          : sw_bytes == 64  ? CU_TENSOR_MAP_SWIZZLE_64B
                          : sw_bytes == 32  ? CU_TENSOR_MAP_SWIZZLE_32B : CU_TENSOR_MAP_SWIZZLE_NONE;
    cuuint64_t dims[2] = {d0, d1};
    cuuint64_t strides[1] = {ld * (uint64_t)elem_bytes};
    cuuint32_t box[2] = {b0, b1};
    cuuint32_t estr[2] = {1, 1};
    alignas(64) CUtensorMap tm;
    CUresult r = c->encode(&tm, elem_bytes == 1 ? CU_TENSOR_MAP_DATA_TYPE_UINT8 : CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<void*>(ptr), dims, strides, box, estr,
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
constexpr int GEMM_STG_BYTES = 4096;                           // per epilogue warp (see stg_f32 / stg_b16)
constexpr int GEMM_THREADS = 576;                              // TMA, MMA, 4 x 4 epilogue warps

template <int BLOCK_N, int STAGES, bool SPLIT>
struct GemmCfg {
    static constexpr int A_BYTES = GEMM_BM * GEMM_BK * 2;            // 16 KB per A term
    static constexpr int B_BYTES = BLOCK_N * GEMM_BK * 2;
    static constexpr int STAGE_BYTES = A_BYTES * (SPLIT ? 2 : 1) + B_BYTES;
    static constexpr int SMEM_BYTES = STAGES * STAGE_BYTES + 16 * GEMM_STG_BYTES + 1024;   // ring + staging + alignment slack
    static constexpr int TMEM_COLS = 2 * BLOCK_N < 32 ? 32 : 2 * BLOCK_N;   // two accumulator buffers (power of 2)
};

// ---- per-warp staging tile (4 KB of shared memory): the epilogue thread owns one ROW of the accumulator, so direct
// global stores touch 32 different 128-byte lines per instruction (measured: ~1.6 TB/s for the whole GPU whatever
// the output type).  Results (and the fp32 residual on the way in) go through this tile instead, so that every
// global access of a warp covers whole 64- or 128-byte row segments.  Layouts, 16-byte pieces XOR-swizzled so that
// both the row-wise (thread = row) and the coalesced (4 or 8 lanes per row) accesses are bank-conflict free:
//   fp32: [32 rows][8 pieces of 4 floats]   piece p of row r at  r * 128 + ((p ^ (r & 7)) << 4)
//   bf16: [32 rows][4 pieces of 8 bf16], hi at +0 and lo at +2048:  r * 64 + ((p ^ ((r >> 1) & 3)) << 4)
__device__ __forceinline__ uint8_t* stg_f32(uint8_t* stg, int r, int p) { return stg + r * 128 + ((p ^ (r & 7)) << 4); }
__device__ __forceinline__ uint8_t* stg_b16(uint8_t* stg, int r, int p) { return stg + r * 64 + ((p ^ ((r >> 1) & 3)) << 4); }

// coalesced copy between the staging tile and global rows: local row rr lives at global row __shfl(row, rr) (< 0: skip)
template <bool LOAD>
__device__ __forceinline__ void stg_copy_f32(uint8_t* stg, float* g, int64_t ld, int col0, int row, int lane) {
#pragma unroll
    for (int i = 0; i < 8; ++i) {                       // 4 rows x 128 B per instruction
        const int rr = 4 * i + (lane >> 3), p = lane & 7;
        const int grow = __shfl_sync(0xffffffffu, row, rr);
        if (grow >= 0) {
            float4* gp = reinterpret_cast<float4*>(g + (int64_t)grow * ld + col0) + p;
            float4* sp = reinterpret_cast<float4*>(stg_f32(stg, rr, p));
            if (LOAD) *sp = *gp; else *gp = *sp;
        }
    }
}
// The bf16 flush with everything that does not depend on the column group precomputed once per tile (the epilogue is issue
// bound: the 64-bit row offsets and the four shuffles were ~ 20 instructions per 8-row store): goff[i] = element offset of
// this lane's piece of local row 8 i + lane / 4 (< 0: skip), soff[i] = its byte offset in the staging tile.
struct FlushB16 { int64_t goff[4]; int soff[4]; };
__device__ __forceinline__ FlushB16 stg_flush_b16_setup(int64_t ld, int row, int lane) {
    FlushB16 f;
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const int rr = 8 * i + (lane >> 2), p = lane & 3;
        const int grow = __shfl_sync(0xffffffffu, row, rr);
        f.goff[i] = grow >= 0 ? (int64_t)grow * ld + p * 8 : -1;
        f.soff[i] = rr * 64 + ((p ^ ((rr >> 1) & 3)) << 4);
    }
    return f;
}
__device__ __forceinline__ void stg_flush_b16(uint8_t* stg, bf16* g, int col0, const FlushB16& f) {
#pragma unroll
    for (int i = 0; i < 4; ++i)                         // 8 rows x 64 B per instruction
        if (f.goff[i] >= 0) *reinterpret_cast<uint4*>(g + f.goff[i] + col0) = *reinterpret_cast<uint4*>(stg + f.soff[i]);
}

// epilogue of one 16-column chunk held in registers (thread = lane = one row); bias_s = this chunk's bias in shared
// memory; cc = 0 / 1: which half of the 32-column staging group; results are left in the staging tile
template <int ACT>
__device__ __forceinline__ void gemm_epilogue_chunk(const uint32_t (&acc)[16], const Epi& ep, const float* bias_s, uint8_t* stg,
                                                    int lane, int cc, float* ss = nullptr, float col_scale = 1.0f) {
    float2 v[8];
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        const float4 b = *reinterpret_cast<const float4*>(bias_s + 4 * j);      // broadcast LDS.128 (zeros when there is no bias)
        const float2 sc = make_float2(ep.out_scale * col_scale, ep.out_scale * col_scale);   // (the staged bias carries col_scale already)
        v[2 * j] = ptx::ffma2(make_float2(__uint_as_float(acc[4 * j]), __uint_as_float(acc[4 * j + 1])), sc, make_float2(b.x, b.y));
        v[2 * j + 1] = ptx::ffma2(make_float2(__uint_as_float(acc[4 * j + 2]), __uint_as_float(acc[4 * j + 3])), sc, make_float2(b.z, b.w));
    }
    if (ss) {                                           // sum of squares of the chunk (attention norms, QKV projection)
        float2 q2 = ptx::fmul2(v[0], v[0]);
#pragma unroll
        for (int j = 1; j < 8; ++j) q2 = ptx::ffma2(v[j], v[j], q2);
        *ss += q2.x + q2.y;
    }
#pragma unroll
    for (int j = 0; j < 8; ++j) {
        if (ACT == ACT_GELU) v[j] = gelu2(v[j]);
        if (ACT == ACT_RELU) v[j] = make_float2(fmaxf(v[j].x, 0.0f), fmaxf(v[j].y, 0.0f));
    }
    if (ep.out_f32) {                                   // fp32 result, optionally + fp32 residual staged in the same place
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            float4* sp = reinterpret_cast<float4*>(stg_f32(stg, lane, 4 * cc + j));
            if (ep.residual) {
                const float4 r = *sp;
                v[2 * j] = ptx::fadd2(v[2 * j], make_float2(r.x, r.y));
                v[2 * j + 1] = ptx::fadd2(v[2 * j + 1], make_float2(r.z, r.w));
            }
            *sp = make_float4(v[2 * j].x, v[2 * j].y, v[2 * j + 1].x, v[2 * j + 1].y);
        }
    } else {                                            // bf16 result as hi (+ lo = T(v - hi))
        uint32_t hi[8], lo[8];
#pragma unroll
        for (int j = 0; j < 8; ++j) {
            __nv_bfloat162 h2 = __floats2bfloat162_rn(v[j].x, v[j].y);
            hi[j] = *reinterpret_cast<uint32_t*>(&h2);
            if (ep.out_act_lo) {
                // bf16 -> fp32 is a 16-bit shift: v - hi as two integer ops + one packed subtract
                const float2 d = ptx::fadd2(v[j], make_float2(-__uint_as_float(hi[j] << 16), -__uint_as_float(hi[j] & 0xffff0000u)));
                __nv_bfloat162 l2 = __floats2bfloat162_rn(d.x, d.y);
                lo[j] = *reinterpret_cast<uint32_t*>(&l2);
            }
        }
#pragma unroll
        for (int j = 0; j < 2; ++j) {
            *reinterpret_cast<uint4*>(stg_b16(stg, lane, 2 * cc + j)) = make_uint4(hi[4 * j], hi[4 * j + 1], hi[4 * j + 2], hi[4 * j + 3]);
            if (ep.out_act_lo)
                *reinterpret_cast<uint4*>(stg_b16(stg + 2048, lane, 2 * cc + j)) = make_uint4(lo[4 * j], lo[4 * j + 1], lo[4 * j + 2], lo[4 * j + 3]);
        }
    }
}

// FP8: A and W are e4m3 (one byte per element, 128 elements per 128-byte swizzled row, K = 32 per MMA): the byte
// arithmetic of the stage ring is that of bf16 with K counted in units of 128 bytes; the epilogue rescales (ep.out_scale).
template <int BLOCK_N, int STAGES, bool SPLIT, int ACT, bool FP8 = false>
__global__ void __launch_bounds__(GEMM_THREADS, 1)
k_tc_gemm(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmA_lo,
          const __grid_constant__ CUtensorMap tmB, int M, int N, int K, Epi ep) {
    using Cfg = GemmCfg<BLOCK_N, STAGES, SPLIT>;
    extern __shared__ uint8_t smem_raw[];
    __shared__ uint64_t bars[2 * STAGES + 4];
    __shared__ uint32_t tmem_base_slot;
    __shared__ __align__(16) float bias_s[2][BLOCK_N];

    const int warp = ptx::uniform_warp_idx(), lane = threadIdx.x & 31;
    const int n_tiles_n = N / BLOCK_N;
    const int total_tiles = ((M + GEMM_BM - 1) / GEMM_BM) * n_tiles_n;
    int m_end = M, nc_rows = 0x7fffffff;       // (read from global memory after the set-up, behind grid_dep_wait)
    // tile -> (m tile, n tile) without a division per tile (every epilogue warp walks all of the CTA's tiles and the epilogue
    // is issue bound): (mi, ni) advance by gridDim.x = dq * n_tiles_n + dr
    const int dq = gridDim.x / n_tiles_n, dr = gridDim.x % n_tiles_n;
    const int mi0 = blockIdx.x / n_tiles_n, ni0 = blockIdx.x % n_tiles_n;
    auto advance = [&](int& mi, int& ni) { mi += dq; ni += dr; if (ni >= n_tiles_n) { ni -= n_tiles_n; ++mi; } };
    // tiles without meaningful rows (all three roles skip the same ones)
    auto skip_tile = [&](int m0) {
        if (m0 >= m_end) return true;
        if (ep.group_rows > 0) m0 %= ep.group_rows;           // (a branch, not a select: no division on the one-stack path)
        return m0 >= nc_rows;
    };
    const uint32_t smem_base = (ptx::smem_u32(smem_raw) + 1023u) & ~1023u;
    const uint32_t bar_full = ptx::smem_u32(&bars[0]);
    const uint32_t bar_empty = ptx::smem_u32(&bars[STAGES]);
    const uint32_t bar_acc_full = ptx::smem_u32(&bars[2 * STAGES]);        // [buf]
    const uint32_t bar_acc_empty = ptx::smem_u32(&bars[2 * STAGES + 2]);   // [buf]

    if (warp == 0 && lane == 0) {
        for (int s = 0; s < STAGES; ++s) { ptx::mbar_init(bar_full + 8 * s, 1); ptx::mbar_init(bar_empty + 8 * s, 1); }
        for (int b = 0; b < 2; ++b) { ptx::mbar_init(bar_acc_full + 8 * b, 1); ptx::mbar_init(bar_acc_empty + 8 * b, 8); }
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
    const int num_kb = K / (FP8 ? 2 * GEMM_BK : GEMM_BK);
    // programmatic dependent launch: the set-up above may overlap the previous kernel's tail; nothing below may
    ptx::grid_dep_wait();
    ptx::grid_dep_launch();
    if (ep.group_offsets) m_end = ep.group_offsets[ep.n_groups + 1];            // grouped: rows beyond the last group
    if (ep.nc_dev) nc_rows = __ldg(ep.nc_dev);

    if (warp == 0) {
        // ---------------- TMA producer: the stage ring runs on across tiles
        uint32_t kbg = 0;
        int mi = mi0, ni = ni0;
        for (int tile = blockIdx.x; tile < total_tiles; tile += gridDim.x, advance(mi, ni)) {
            const int m0 = mi * GEMM_BM, n0 = ni * BLOCK_N;
            if (skip_tile(m0)) continue;
            int w_row0 = 0;
            if (ep.group_offsets) {                               // grouped GEMM (per-type embedding weights)
                int g = 1;
                while (g < ep.n_groups && m0 >= ep.group_offsets[g + 1]) ++g;
                w_row0 = (g - 1) * N;
            } else if (ep.group_rows > 0) w_row0 = (m0 / ep.group_rows) * N;   // one weight block per encoder stack
            for (int kb = 0; kb < num_kb; ++kb, ++kbg) {
                const uint32_t s = kbg % STAGES;
                ptx::mbar_wait(bar_empty + 8 * s, ((kbg / STAGES) & 1) ^ 1);
                if (lane == 0) {
                    const uint32_t st = smem_base + s * Cfg::STAGE_BYTES;
                    ptx::mbar_expect_tx(bar_full + 8 * s, Cfg::STAGE_BYTES);
                    constexpr int KE = FP8 ? 2 * GEMM_BK : GEMM_BK;           // elements of K per stage (128 bytes per row)
                    ptx::tma_load_2d(st, &tmA, bar_full + 8 * s, kb * KE, m0);
                    if (SPLIT) ptx::tma_load_2d(st + Cfg::A_BYTES, &tmA_lo, bar_full + 8 * s, kb * KE, m0);
                    ptx::tma_load_2d(st + Cfg::A_BYTES * (SPLIT ? 2 : 1), &tmB, bar_full + 8 * s, kb * KE, w_row0 + n0);
                }
                __syncwarp();
            }
        }
    } else if (warp == 1) {
        // ---------------- MMA issuer (all lanes, warp-uniform operands; one lane elected inside the wrappers)
        constexpr uint32_t idesc = FP8 ? ptx::umma_idesc_e4m3(GEMM_BM, BLOCK_N) : ptx::umma_idesc_bf16(GEMM_BM, BLOCK_N);
        uint32_t kbg = 0;
        int it = 0;
        int mi = mi0, ni = ni0;
        for (int tile = blockIdx.x; tile < total_tiles; tile += gridDim.x, advance(mi, ni)) {
            if (skip_tile(mi * GEMM_BM)) continue;
            const int buf = it & 1;
            ptx::mbar_wait(bar_acc_empty + 8 * buf, ((it >> 1) & 1) ^ 1);      // the epilogue drained this buffer
            ptx::tc_fence_after();
            const uint32_t d_tmem = tmem_base + buf * BLOCK_N;
            for (int kb = 0; kb < num_kb; ++kb, ++kbg) {
                const uint32_t s = kbg % STAGES;
                ptx::mbar_wait(bar_full + 8 * s, (kbg / STAGES) & 1);
                ptx::tc_fence_after();
                const uint32_t a_addr = smem_base + s * Cfg::STAGE_BYTES;
                const uint32_t b_addr = a_addr + Cfg::A_BYTES * (SPLIT ? 2 : 1);
#pragma unroll
                for (int k = 0; k < GEMM_BK / 16; ++k) {
                    const uint64_t bd = ptx::umma_desc_kmajor(b_addr + k * 32, 128);
                    if (FP8) ptx::mma_ss_f8(d_tmem, ptx::umma_desc_kmajor(a_addr + k * 32, 128), bd, idesc, (kb | k) != 0);
                    else ptx::mma_ss(d_tmem, ptx::umma_desc_kmajor(a_addr + k * 32, 128), bd, idesc, (kb | k) != 0);
                    if (SPLIT) ptx::mma_ss(d_tmem, ptx::umma_desc_kmajor(a_addr + Cfg::A_BYTES + k * 32, 128), bd, idesc, 1);
                }
                ptx::mma_commit(bar_empty + 8 * s);               // frees the stage when these MMAs retire
            }
            ptx::mma_commit(bar_acc_full + 8 * buf);
            ++it;
        }
    } else {
        // ---------------- epilogue: 4 warpgroups = (accumulator buffer e) x (column half): 4 warps per SM
        // sub-partition keep the issue-bound activation epilogues busy
        const int ew = warp - 2;
        const int e = (ew >> 2) & 1;
        const int hcol = (ew >> 3) * (BLOCK_N / 2);
        const int q = warp & 3;                                   // TMEM lane quarter this warp may access
        const int tid = ((ew >> 3) * 4 + (ew & 3)) * 32 + lane;   // 0..255 among the threads serving buffer e
        uint8_t* stg = smem_raw + (smem_base - ptx::smem_u32(smem_raw)) + STAGES * Cfg::STAGE_BYTES + ew * GEMM_STG_BYTES;
        int it = 0;
        int mi = mi0, ni = ni0;
        for (int tile = blockIdx.x; tile < total_tiles; tile += gridDim.x, advance(mi, ni)) {
            const int m0 = mi * GEMM_BM, n0 = ni * BLOCK_N;
            if (skip_tile(m0)) continue;
            if ((it & 1) != e) { ++it; continue; }
            int w_row0 = 0;
            if (ep.group_offsets) {
                int g = 1;
                while (g < ep.n_groups && m0 >= ep.group_offsets[g + 1]) ++g;
                w_row0 = (g - 1) * N;
            } else if (ep.group_rows > 0) w_row0 = (m0 / ep.group_rows) * N;
            // this tile's bias -> shared memory (read back as broadcast 128-bit loads)
            asm volatile("bar.sync %0, 256;" ::"r"(1 + e) : "memory");          // everyone is done with the last tile's
            const int q_cols = ep.qn ? ep.nd : 0;                 // columns below it (q of the QKV projection) carry ep.q_scale
            for (int c = tid; c < BLOCK_N; c += 256)
                bias_s[e][c] = ep.bias ? __ldg(ep.bias + w_row0 + n0 + c) * (n0 + c < q_cols ? ep.q_scale : 1.0f) : 0.0f;
            asm volatile("bar.sync %0, 256;" ::"r"(1 + e) : "memory");
            const int m = m0 + q * 32 + lane;
            const bool row_ok = m < M;
            int row = m;
            if (row_ok && ep.row_perm) row = ep.row_perm[m];
            const bool write_ok = row_ok && row >= 0;
            ptx::mbar_wait_long(bar_acc_full + 8 * e, (it >> 1) & 1);   // (suspends: a spinning warp takes issue slots from the working ones)
            ptx::tc_fence_after();
            const uint32_t t_addr = tmem_base + ((uint32_t)(q * 32) << 16) + e * BLOCK_N + hcol;
            const int srow = write_ok ? row : -1;                 // destination row of this lane's accumulator row
            const FlushB16 fl = stg_flush_b16_setup(ep.ld_act, srow, lane);   // (bf16 outputs; unused for fp32 ones)
            uint32_t ra[16], rb[16];
            ptx::tmem_ld16(t_addr, ra);
            // attention norms (QKV projection): this lane's row, its event, running sum of squares of the current head
            const bool norms = ep.qn != nullptr && n0 + hcol < 2 * ep.nd;
            int n_ev = -1;
            if (norms && row_ok) {
                int mg = m;
                if (ep.group_rows > 0) mg %= ep.group_rows;
                if (mg < nc_rows) n_ev = __ldg(ep.row_event + m);
            }
            float n_ss = 0.0f;
            // (no runtime division in this epilogue: the head width is a power of two, q | k | v by comparison)
            const int hd_shift = 31 - __clz(ep.nhd | 1);
            auto norm_emit = [&](int col_end) {                   // columns up to col_end (exclusive) close a head
                if (col_end & (ep.nhd - 1)) return;
                const int blk = col_end > ep.nd ? 1 : 0, head = (col_end - 1 - blk * ep.nd) >> hd_shift;
                const float nrm = sqrtf(n_ss);
                n_ss = 0.0f;
                if (blk == 0) { if (n_ev >= 0) ep.qn[(int64_t)m * ep.nH + head] = nrm; }
                else {
                    const unsigned grp = __match_any_sync(0xffffffffu, n_ev);
                    const unsigned mx = __reduce_max_sync(grp, __float_as_uint(nrm));
                    if (n_ev >= 0 && (int)(threadIdx.x & 31) == __ffs(grp) - 1)
                        atomicMax(reinterpret_cast<unsigned*>(ep.kmax) + (int64_t)n_ev * ep.nH + head, mx);
                }
            };
#pragma unroll
            for (int c = 0; c < BLOCK_N / 2; c += 32) {           // one 32-column staging group per iteration
                const int col0 = n0 + hcol + c;
                if (ep.residual) stg_copy_f32<true>(stg, const_cast<float*>(ep.residual), ep.ld_res, col0, srow, lane);
                ptx::tmem_ld_wait();
                ptx::tmem_ld16(t_addr + c + 16, rb);
                __syncwarp();
                const float cs0 = col0 < q_cols ? ep.q_scale : 1.0f, cs1 = col0 + 16 < q_cols ? ep.q_scale : 1.0f;
                gemm_epilogue_chunk<ACT>(ra, ep, &bias_s[e][hcol + c], stg, lane, 0, norms ? &n_ss : nullptr, cs0);
                if (norms) norm_emit(col0 + 16);
                ptx::tmem_ld_wait();
                if (c + 32 < BLOCK_N / 2) ptx::tmem_ld16(t_addr + c + 32, ra);
                gemm_epilogue_chunk<ACT>(rb, ep, &bias_s[e][hcol + c + 16], stg, lane, 1, norms ? &n_ss : nullptr, cs1);
                if (norms) norm_emit(col0 + 32);
                __syncwarp();
                if (ep.out_f32) {
                    stg_copy_f32<false>(stg, ep.out_f32, ep.ld_f32, col0, srow, lane);
                } else {
                    stg_flush_b16(stg, (bf16*)ep.out_act, col0, fl);
                    if (ep.out_act_lo) stg_flush_b16(stg + 2048, (bf16*)ep.out_act_lo, col0, fl);
                }
                __syncwarp();
            }
            ptx::tc_fence_before();
            __syncwarp();
            if (lane == 0) ptx::mbar_arrive(bar_acc_empty + 8 * e);
            ++it;
        }
    }
    ptx::tc_fence_before();
    __syncthreads();
    if (warp == 1) ptx::tmem_dealloc(tmem_base, Cfg::TMEM_COLS);
}

// ------------------------------------------------------------------------------------------------ launch
template <int BLOCK_N, int STAGES, bool SPLIT, int ACT, bool FP8 = false>
static int tc_gemm_launch_act(TcContext* c, const bf16* A, const bf16* A_lo, const bf16* W, int M, int N, int K,
                              int w_rows, const Epi& ep, cudaStream_t st) {
    using Cfg = GemmCfg<BLOCK_N, STAGES, SPLIT>;
    CUtensorMap tmA, tmAlo, tmB;
    constexpr int EB = FP8 ? 1 : 2, KE = FP8 ? 2 * GEMM_BK : GEMM_BK;
    if (tc_tensor_map(c, &tmA, A, K, M, K, KE, GEMM_BM, EB)) return -1;
    if (SPLIT) { if (tc_tensor_map(c, &tmAlo, A_lo, K, M, K, KE, GEMM_BM, EB)) return -1; }
    else tmAlo = tmA;
    if (tc_tensor_map(c, &tmB, W, K, w_rows, K, KE, BLOCK_N, EB)) return -1;
    auto kern = k_tc_gemm<BLOCK_N, STAGES, SPLIT, ACT, FP8>;
    if (tc_set_smem_attr(c, (const void*)kern, Cfg::SMEM_BYTES)) return -1;
    const int total_tiles = ((M + GEMM_BM - 1) / GEMM_BM) * (N / BLOCK_N);
    const int grid = total_tiles < c->num_sms ? total_tiles : c->num_sms;
    tc_launch(kern, dim3(grid), dim3(GEMM_THREADS), Cfg::SMEM_BYTES, st, c->pdl, tmA, tmAlo, tmB, M, N, K, ep);
    return 0;
}

template <int BLOCK_N, int STAGES, bool SPLIT>
static int tc_gemm_launch_cfg(TcContext* c, const bf16* A, const bf16* A_lo, const bf16* W, int M, int N, int K,
                              int w_rows, const Epi& ep, cudaStream_t st) {
    switch (ep.act) {                                 // the activation is compiled into the epilogue
        case ACT_GELU: return tc_gemm_launch_act<BLOCK_N, STAGES, SPLIT, ACT_GELU>(c, A, A_lo, W, M, N, K, w_rows, ep, st);
        case ACT_RELU: return tc_gemm_launch_act<BLOCK_N, STAGES, SPLIT, ACT_RELU>(c, A, A_lo, W, M, N, K, w_rows, ep, st);
    }
    return tc_gemm_launch_act<BLOCK_N, STAGES, SPLIT, ACT_NONE>(c, A, A_lo, W, M, N, K, w_rows, ep, st);
}

int tc_gemm_launch(TcContext* c, const bf16* A, const bf16* A_lo, const bf16* W, int M, int N, int K,
                          const Epi& ep, cudaStream_t st) {
    if (ep.out_f32 ? (ep.out_act != nullptr) : (ep.out_act == nullptr || ep.residual != nullptr)) {
        snprintf(c->err, sizeof c->err, "tc_gemm: the epilogue writes either fp32 (+ residual) or bf16 hi (+ lo)"); return -1;
    }
    if (N % 64 || K % 64) { snprintf(c->err, sizeof c->err, "tc_gemm: N=%d, K=%d must be multiples of 64", N, K); return -1; }
    const int w_rows = (ep.group_offsets || ep.group_rows > 0) ? ep.n_groups * N : N;
    if (N % 128 == 0) {
        return A_lo ? tc_gemm_launch_cfg<128, 3, true>(c, A, A_lo, W, M, N, K, w_rows, ep, st)
                    : tc_gemm_launch_cfg<128, 4, false>(c, A, nullptr, W, M, N, K, w_rows, ep, st);
    }
    return A_lo ? tc_gemm_launch_cfg<64, 3, true>(c, A, A_lo, W, M, N, K, w_rows, ep, st)
                : tc_gemm_launch_cfg<64, 5, false>(c, A, nullptr, W, M, N, K, w_rows, ep, st);
}

// C = (A W^T) out_scale + bias ...: A [M, K] and W [N, K] are e4m3 bytes (kind::f8f6f4), K % 128 == 0, N % 128 == 0;
// no activation, no split (the QKV projection, NEXT-3).
int tc_gemm_fp8_launch(TcContext* c, const uint8_t* A, const uint8_t* W, int M, int N, int K, const Epi& ep, cudaStream_t st) {
    if (N % 128 || K % 128 || ep.act != ACT_NONE) { snprintf(c->err, sizeof c->err, "tc_gemm_fp8: N=%d, K=%d must be multiples of 128, no activation", N, K); return -1; }
    if (ep.out_f32 ? (ep.out_act != nullptr) : (ep.out_act == nullptr || ep.residual != nullptr)) {
        snprintf(c->err, sizeof c->err, "tc_gemm_fp8: the epilogue writes either fp32 (+ residual) or bf16 hi (+ lo)"); return -1;
    }
    const int w_rows = (ep.group_offsets || ep.group_rows > 0) ? ep.n_groups * N : N;
    return tc_gemm_launch_act<128, 4, false, ACT_NONE, true>(c, (const bf16*)A, nullptr, (const bf16*)W, M, N, K, w_rows, ep, st);
}

}  // namespace mlpf
