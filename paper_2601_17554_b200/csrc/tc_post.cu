// tc_post.cu -- the whole post-attention half of an encoder block as ONE tcgen05 / TMEM / TMA kernel (sm_100a):
//
//   h1 = h + o Wo^T + bo            (a5: output projection + residual, PAPER.md L148 / L156)
//   u2 = LN2(h1)                    (a5's epilogue: pre-LN of the FFN, L156 + reading A7/A8)
//   g  = act(u2 W1^T + b1)          (a6: FFN first linear + activation, L156 + A5/A6)
//   h2 = h1 + g W2^T + b2           (a7: FFN second linear + residual)
//   u' = LN_next(h2)                (a7's epilogue: the NEXT block's LN1, or the final LN before the heads)
//
// Neither u2 nor the dff-wide hidden g ever reaches HBM: per 128-row tile the CTA keeps o (then u2) as a resident
// shared-memory A operand (bf16 hi + lo), streams Wo / W1 / W2 through a TMA ring, and chains the MMAs through TMEM:
//   TMEM columns [0, D)        acc: o Wo^T, then (rewritten as h1 by the epilogue) the accumulator of FFN2, so that the
//                              residual add of a7 is the accumulator's initial value;
//   TMEM columns 256 + 128 b   S_b (b = 0, 1): one 128-column chunk of u2 W1^T, double-buffered.  The epilogue warps read
//                              a chunk, add b1, apply the activation and write the result BACK over the same columns as
//                              packed bf16 (hi | lo per 32-column group), which the second MMA takes as its A operand
//                              straight from TMEM (same mechanism as P in the attention kernel).
// D = d_model in {64, 128, 256} (a full row per CTA, which is what lets both LayerNorms live in epilogues; d = 512
// needs 512 accumulator columns and keeps the unfused chain).  dff % 128 == 0.
//
// Warps: 0 = TMA producer, 1 = MMA issuer (all lanes run the issue code, one lane elected inside the wrappers),
// 2..17 = 16 epilogue warps = (TMEM lane quarter q = warp % 4) x (column group cg): thread = one row of the tile.
// LayerNorm statistics: every warp takes (mean, centred second moment) of its D/4 columns exactly (two passes over
// registers) and the four column groups of a row are merged with the pairwise formula, so there is no E[x^2] - mean^2.
// Grouped mode (two parallel encoders, L156): tile m0 uses weight / vector block m0 / group_rows.
#include "tc_api.h"
#include "ptx.cuh"
#include "epi_math.cuh"
#include <cuda_fp8.h>

namespace mlpf {

constexpr int POST_BM = 128, POST_CH = 128, POST_SLOT = 16384, POST_THREADS = 576;

template <int D>
struct PostCfg {
    static constexpr int KB = D / 64;                     // 64-wide k-blocks of the D-wide operands (o, u2)
    static constexpr int NB = D < 128 ? D : 128;          // N of the MMAs that produce D columns
    static constexpr int NH = D / NB;
    static constexpr int A_BYTES = 2 * KB * POST_SLOT;    // hi + lo
    static constexpr int NS = D == 256 ? 5 : 6;           // ring slots of 16 KB
    static constexpr int CW = D / 4;                      // columns of a row owned by one epilogue warp
    static constexpr int PIECE = CW < 32 ? CW : 32;
    static constexpr int PART_BYTES = 4 * POST_BM * 8;
    static int smem_bytes(int dff) { return A_BYTES + NS * POST_SLOT + PART_BYTES + (6 * D + dff) * 4 + 1024; }
};

struct PostParams {
    int M, dff, group_rows;
    const int* nc_dev;              // meaningful rows (per group), device, may be null: tiles at or beyond it are skipped
    const float *bo, *ln2g, *ln2b, *b1, *b2, *lnng, *lnnb;   // per group: D, D, D, dff, D, D, D floats
    float eps;
    float* h;                       // [M, D] fp32 residual stream, updated in place
    int h_in_tiled, h_out_tiled;    // layout of h on the way in / out: 0 = row-major, 1 = tiled (see h_off)
    bf16* u_out; bf16* u_out_lo;    // [M, D] next LayerNorm output (lo may be null)
    uint8_t* u_out_f8; float f8_scale;   // optional e4m3 copy of it times f8_scale (FP8 operands of the next QKV projection)
    int next_ln;                    // 0: u_out = T(h2) (final_ln = 0)
    bf16* dbg_u2; bf16* dbg_g;      // debug taps (null in production): u2 [M, D], g [M, dff] (hi terms)
};

// The epilogue thread owns one ROW of the tile, so 16-byte accesses to a row-major [M, D] matrix touch 32 different
// 128-byte lines per warp instruction (one L1TEX wavefront each: measured 11 k cycles per 128 x 256 fp32 tile, with
// the tensor pipe idle).  The residual stream is private to the library's kernels, so between fused blocks it lives in
// a TILED layout in which those accesses are contiguous: element (row, col) of 128-row tile t = row / 128 is at
//   t * 128 * D + (col / 4) * 512 + (row % 128) * 4 + col % 4        (floats)
// i.e. for each group of 4 columns the 128 rows of the tile are adjacent: a warp's LDG.128 / STG.128 covers 512
// contiguous bytes.  The block reads either layout and writes either layout (first block: row-major in, tiled out);
// a tiled buffer holds whole 128-row tiles.
// Both layouts as (base, stride): the float4 holding columns 4 k .. 4 k + 3 of row r of tile t is at base + k * stride.
template <int D>
__device__ __forceinline__ void h_addr(bool tiled, int tile, int r, int64_t& base, int& stride) {
    base = tiled ? (int64_t)tile * (POST_BM * D) + r * 4 : ((int64_t)tile * POST_BM + r) * D;
    stride = tiled ? POST_BM * 4 : 4;
}

template <int N> __device__ __forceinline__ void tmem_ld_n(uint32_t addr, uint32_t (&r)[N]);
template <> __device__ __forceinline__ void tmem_ld_n<32>(uint32_t addr, uint32_t (&r)[32]) { ptx::tmem_ld32(addr, r); }
template <> __device__ __forceinline__ void tmem_ld_n<16>(uint32_t addr, uint32_t (&r)[16]) { ptx::tmem_ld16(addr, r); }
template <int N> __device__ __forceinline__ void tmem_st_n(uint32_t addr, const uint32_t (&r)[N]) {
#pragma unroll
    for (int i = 0; i < N / 16; ++i) ptx::tmem_st16(addr + 16 * i, *reinterpret_cast<const uint32_t(*)[16]>(&r[16 * i]));
}

__device__ __forceinline__ void st_global_v8(void* ptr, const uint32_t* v) {
    asm volatile("st.global.v8.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8};" ::"l"(ptr), "r"(v[0]), "r"(v[1]), "r"(v[2]), "r"(v[3]),
                 "r"(v[4]), "r"(v[5]), "r"(v[6]), "r"(v[7]) : "memory");
}

// (n, mean, M2) of a set merged with (nb, mb, m2b) of another (Chan et al.): exact pairwise update
__device__ __forceinline__ void stats_merge(float& n, float& mean, float& m2, float nb, float mb, float m2b) {
    const float nn = n + nb, delta = mb - mean;
    mean += delta * (nb / nn);
    m2 += m2b + delta * delta * (n * nb / nn);
    n = nn;
}
template <int N>
__device__ __forceinline__ void stats_piece(const float (&v)[N], float& n, float& mean, float& m2) {
    float s[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
    for (int i = 0; i < N; ++i) s[i & 3] += v[i];
    const float pm = ((s[0] + s[1]) + (s[2] + s[3])) * (1.0f / N);
    float q[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
    for (int i = 0; i < N; ++i) { const float c = v[i] - pm; q[i & 3] = fmaf(c, c, q[i & 3]); }
    const float pq = (q[0] + q[1]) + (q[2] + q[3]);
    if (n == 0.0f) { n = (float)N; mean = pm; m2 = pq; }
    else stats_merge(n, mean, m2, (float)N, pm, pq);
}

template <int D, int ACT>
__global__ void __launch_bounds__(POST_THREADS, 1)
k_tc_post(const __grid_constant__ CUtensorMap tmO, const __grid_constant__ CUtensorMap tmOlo,
          const __grid_constant__ CUtensorMap tmWo, const __grid_constant__ CUtensorMap tmW1,
          const __grid_constant__ CUtensorMap tmW2, PostParams p) {
    using Cfg = PostCfg<D>;
    constexpr int KB = Cfg::KB, NB = Cfg::NB, NH = Cfg::NH, NS = Cfg::NS, CW = Cfg::CW, PIECE = Cfg::PIECE;
    extern __shared__ uint8_t smem_raw[];
    __shared__ uint64_t bars[2 * NS + 11];
    __shared__ uint32_t tmem_base_slot;

    const int warp = ptx::uniform_warp_idx(), lane = threadIdx.x & 31;
    const int n_tiles = (p.M + POST_BM - 1) / POST_BM;
    const int NC = p.dff / POST_CH;
    int nc_rows = 0x7fffffff;                  // (read after the set-up, behind grid_dep_wait)
    auto skip_tile = [&](int tile) { return (tile * POST_BM) % p.group_rows >= nc_rows; };   // all three roles skip the same tiles
    const uint32_t smem_base = (ptx::smem_u32(smem_raw) + 1023u) & ~1023u;
    uint8_t* const smem_gen = smem_raw + (smem_base - ptx::smem_u32(smem_raw));
    const uint32_t sA = smem_base, sRing = sA + Cfg::A_BYTES;
    float2* const part = reinterpret_cast<float2*>(smem_gen + Cfg::A_BYTES + NS * POST_SLOT);
    float* const vec = reinterpret_cast<float*>(smem_gen + Cfg::A_BYTES + NS * POST_SLOT + Cfg::PART_BYTES);
    const uint32_t bar_full = ptx::smem_u32(&bars[0]), bar_empty = ptx::smem_u32(&bars[NS]);
    const uint32_t bar_a_full = ptx::smem_u32(&bars[2 * NS]), bar_a_free = bar_a_full + 8, bar_acc_full = bar_a_full + 16,
                   bar_u2 = bar_a_full + 24, bar_s_full = bar_a_full + 32 /* [2] */, bar_g = bar_a_full + 48 /* [2] */,
                   bar_acc_final = bar_a_full + 64, bar_acc_free = bar_a_full + 72;

    if (warp == 0 && lane == 0) {
        for (int s = 0; s < NS; ++s) { ptx::mbar_init(bar_full + 8 * s, 1); ptx::mbar_init(bar_empty + 8 * s, 1); }
        ptx::mbar_init(bar_a_full, 1); ptx::mbar_init(bar_a_free, 1); ptx::mbar_init(bar_acc_full, 1);
        ptx::mbar_init(bar_u2, 16);
        for (int b = 0; b < 2; ++b) { ptx::mbar_init(bar_s_full + 8 * b, 1); ptx::mbar_init(bar_g + 8 * b, 16); }
        ptx::mbar_init(bar_acc_final, 1); ptx::mbar_init(bar_acc_free, 16);
        ptx::fence_barrier_init();
        ptx::tma_prefetch_desc(&tmO); ptx::tma_prefetch_desc(&tmOlo); ptx::tma_prefetch_desc(&tmWo);
        ptx::tma_prefetch_desc(&tmW1); ptx::tma_prefetch_desc(&tmW2);
    }
    if (warp == 1) {
        ptx::tmem_alloc(ptx::smem_u32(&tmem_base_slot), 512);
        ptx::tmem_relinquish();
    }
    ptx::tc_fence_before();
    __syncthreads();
    ptx::tc_fence_after();
    const uint32_t tmem_base = tmem_base_slot;
    // programmatic dependent launch: the set-up above may overlap the previous kernel's tail; nothing below may
    ptx::grid_dep_wait();
    ptx::grid_dep_launch();
    if (p.nc_dev) nc_rows = __ldg(p.nc_dev);

    if (warp == 0) {
        // ------------------------------------------------------------ TMA producer: loads in exactly the issuer's order
        uint32_t slot_it = 0;
        auto load_b = [&](const CUtensorMap* tm, int k0, int row0, uint32_t bytes) {
            const uint32_t s = slot_it % NS;
            ptx::mbar_wait(bar_empty + 8 * s, ((slot_it / NS) & 1) ^ 1);
            if (lane == 0) {
                ptx::mbar_expect_tx(bar_full + 8 * s, bytes);
                ptx::tma_load_2d(sRing + s * POST_SLOT, tm, bar_full + 8 * s, k0, row0);
            }
            __syncwarp();
            ++slot_it;
        };
        int it = -1;
        for (int tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
            if (skip_tile(tile)) continue;
            ++it;
            const int m0 = tile * POST_BM, g = m0 / p.group_rows;
            if (it > 0) ptx::mbar_wait(bar_a_free, (it - 1) & 1);        // the last tile's u2 is no longer read
            if (lane == 0) {
                ptx::mbar_expect_tx(bar_a_full, Cfg::A_BYTES);
                for (int kb = 0; kb < KB; ++kb) {
                    ptx::tma_load_2d(sA + kb * POST_SLOT, &tmO, bar_a_full, kb * 64, m0);
                    ptx::tma_load_2d(sA + (KB + kb) * POST_SLOT, &tmOlo, bar_a_full, kb * 64, m0);
                }
            }
            __syncwarp();
            for (int kb = 0; kb < KB; ++kb)
                for (int nh = 0; nh < NH; ++nh) load_b(&tmWo, kb * 64, g * D + nh * NB, NB * 128);
            auto load_w1 = [&](int c) { for (int kb = 0; kb < KB; ++kb) load_b(&tmW1, kb * 64, g * p.dff + c * POST_CH, POST_SLOT); };
            auto load_w2 = [&](int c) {
                for (int kb2 = 0; kb2 < 2; ++kb2)
                    for (int nh = 0; nh < NH; ++nh) load_b(&tmW2, c * POST_CH + kb2 * 64, g * D + nh * NB, NB * 128);
            };
            load_w1(0);
            if (NC > 1) load_w1(1);
            for (int c = 0; c < NC; ++c) {
                load_w2(c);
                if (c + 2 < NC) load_w1(c + 2);
            }
        }
    } else if (warp == 1) {
        // ------------------------------------------------------------ MMA issuer
        constexpr uint32_t idesc_d = ptx::umma_idesc_bf16(POST_BM, NB);
        constexpr uint32_t idesc_s = ptx::umma_idesc_bf16(POST_BM, POST_CH);
        uint32_t slot_it = 0, ph_g = 0;
        auto wait_slot = [&]() -> uint32_t {
            const uint32_t s = slot_it % NS;
            ptx::mbar_wait(bar_full + 8 * s, (slot_it / NS) & 1);
            ptx::tc_fence_after();
            return sRing + s * POST_SLOT;
        };
        auto free_slot = [&]() { ptx::mma_commit(bar_empty + 8 * (slot_it % NS)); ++slot_it; };
        int it = -1;
        for (int tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
            if (skip_tile(tile)) continue;
            ++it;
            ptx::mbar_wait(bar_a_full, it & 1);
            if (it > 0) ptx::mbar_wait(bar_acc_free, (it - 1) & 1);      // the last tile's final epilogue drained acc
            ptx::tc_fence_after();
            // acc = o Wo^T (hi + lo)
            for (int kb = 0; kb < KB; ++kb)
                for (int nh = 0; nh < NH; ++nh) {
                    const uint32_t b = wait_slot();
#pragma unroll
                    for (int k = 0; k < 4; ++k) {
                        const uint64_t bd = ptx::umma_desc_kmajor(b + k * 32, 128);
                        ptx::mma_ss(tmem_base + nh * NB, ptx::umma_desc_kmajor(sA + kb * POST_SLOT + k * 32, 128), bd, idesc_d, (kb | k) != 0);
                        ptx::mma_ss(tmem_base + nh * NB, ptx::umma_desc_kmajor(sA + (KB + kb) * POST_SLOT + k * 32, 128), bd, idesc_d, 1);
                    }
                    free_slot();
                }
            ptx::mma_commit(bar_acc_full);
            ptx::mbar_wait(bar_u2, it & 1);                              // u2 in shared memory, h1 in acc
            ptx::tc_fence_after();
            auto mma1 = [&](int c) {                                     // S_(c&1) = u2 W1[chunk c]^T
                const uint32_t sb = tmem_base + 256 + 128 * (c & 1);
                for (int kb = 0; kb < KB; ++kb) {
                    const uint32_t b = wait_slot();
#pragma unroll
                    for (int k = 0; k < 4; ++k) {
                        const uint64_t bd = ptx::umma_desc_kmajor(b + k * 32, 128);
                        ptx::mma_ss(sb, ptx::umma_desc_kmajor(sA + kb * POST_SLOT + k * 32, 128), bd, idesc_s, (kb | k) != 0);
                        ptx::mma_ss(sb, ptx::umma_desc_kmajor(sA + (KB + kb) * POST_SLOT + k * 32, 128), bd, idesc_s, 1);
                    }
                    free_slot();
                }
                ptx::mma_commit(bar_s_full + 8 * (c & 1));
            };
            mma1(0);
            if (NC > 1) mma1(1);
            if (NC <= 2) ptx::mma_commit(bar_a_free);
            for (int c = 0; c < NC; ++c) {
                const int bsel = c & 1;
                ptx::mbar_wait(bar_g + 8 * bsel, (ph_g >> bsel) & 1);    // g(c) is in TMEM over S_(c&1)
                ph_g ^= 1u << bsel;
                ptx::tc_fence_after();
                const uint32_t gb = tmem_base + 256 + 128 * bsel;
                for (int kb2 = 0; kb2 < 2; ++kb2)                        // acc += g(c) W2[:, chunk c]^T (hi + lo)
                    for (int nh = 0; nh < NH; ++nh) {
                        const uint32_t b = wait_slot();
#pragma unroll
                        for (int k = 0; k < 4; ++k) {
                            const int j = kb2 * 4 + k;                   // 16-wide k-step of the chunk = 8 packed columns
                            const uint64_t bd = ptx::umma_desc_kmajor(b + k * 32, 128);
                            const uint32_t a_hi = gb + 32 * (j >> 1) + 8 * (j & 1);
                            ptx::mma_ts(tmem_base + nh * NB, a_hi, bd, idesc_d, 1);
                            ptx::mma_ts(tmem_base + nh * NB, a_hi + 16, bd, idesc_d, 1);
                        }
                        free_slot();
                    }
                if (c + 2 < NC) {                                        // S_(c&1) is reused: in order after the MMAs above
                    mma1(c + 2);
                    if (c + 3 == NC) ptx::mma_commit(bar_a_free);        // that was the last reader of u2
                }
            }
            ptx::mma_commit(bar_acc_final);
        }
    } else {
        // ------------------------------------------------------------ epilogue warps
        const int ew = warp - 2, q = warp & 3, cg = ew >> 2;
        const int et = ew * 32 + lane;                    // 0..511
        const int r = q * 32 + lane;                      // row of the tile
        const uint32_t lane_addr = tmem_base + ((uint32_t)(q * 32) << 16);
        float* const v_bo = vec; float* const v_g2 = vec + D; float* const v_b2ln = vec + 2 * D;
        float* const v_b2 = vec + 3 * D; float* const v_gn = vec + 4 * D; float* const v_bn = vec + 5 * D;
        float* const v_b1 = vec + 6 * D;
        uint32_t ph_s = 0;
        int it = -1, g_staged = -1;
        // mean and 1/sigma of the row from the four column groups' partials (each over CW columns)
        auto row_stats = [&](float n, float mean, float m2, float& mu, float& rstd) {
            part[cg * POST_BM + r] = make_float2(mean, m2);
            asm volatile("bar.sync %0, 128;" ::"r"(2 + q) : "memory");
            float tn = 0.f, tm = 0.f, t2 = 0.f;
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                const float2 pk = part[k * POST_BM + r];
                if (k == 0) { tn = n; tm = pk.x; t2 = pk.y; }
                else stats_merge(tn, tm, t2, n, pk.x, pk.y);
            }
            asm volatile("bar.sync %0, 128;" ::"r"(2 + q) : "memory");   // everyone has read: `part` may be rewritten
            mu = tm;
            rstd = rsqrtf(t2 * (1.0f / D) + p.eps);
        };
        for (int tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
            if (skip_tile(tile)) continue;
            ++it;
            const int m0 = tile * POST_BM, g = m0 / p.group_rows;
            const int row = m0 + r;
            const bool row_ok = row < p.M;
            // this tile's vectors (per group) -> shared memory; they change only where the group (encoder stack) does
            if (g != g_staged) {
                asm volatile("bar.sync 1, 512;" ::: "memory");
                for (int i = et; i < D; i += 512) {
                    v_bo[i] = __ldg(p.bo + g * D + i); v_g2[i] = __ldg(p.ln2g + g * D + i); v_b2ln[i] = __ldg(p.ln2b + g * D + i);
                    v_b2[i] = __ldg(p.b2 + g * D + i);
                    v_gn[i] = p.next_ln ? __ldg(p.lnng + g * D + i) : 1.0f; v_bn[i] = p.next_ln ? __ldg(p.lnnb + g * D + i) : 0.0f;
                }
                for (int i = et; i < p.dff; i += 512) v_b1[i] = __ldg(p.b1 + g * p.dff + i);
                asm volatile("bar.sync 1, 512;" ::: "memory");
                g_staged = g;
            }

            // ---------------- epilogue of the output projection: h1 = h + acc + bo -> acc (TMEM); u2 = LN2(h1) -> A operand
            float sn = 0.f, smean = 0.f, sm2 = 0.f;
            // rows past M (last tile) read the last valid row instead (their results are never stored): the loads need
            // no predicate or branch, so all of a piece's loads are in flight together
            const int r_ld = min(r, p.M - 1 - m0);
            int64_t hin_base, hout_base; int hin_stride, hout_stride;
            h_addr<D>(p.h_in_tiled != 0, tile, r_ld, hin_base, hin_stride);
            h_addr<D>(p.h_out_tiled != 0, tile, r, hout_base, hout_stride);
            // the residual rows of the first piece are fetched while the output projection's MMAs still run
            float4 hv0[PIECE / 4];
#pragma unroll
            for (int i = 0; i < PIECE / 4; ++i)
                hv0[i] = *reinterpret_cast<const float4*>(p.h + hin_base + (int64_t)(cg * CW / 4 + i) * hin_stride);
            ptx::mbar_wait(bar_acc_full, it & 1);
            ptx::tc_fence_after();
#pragma unroll
            for (int c0 = cg * CW; c0 < (cg + 1) * CW; c0 += PIECE) {
                uint32_t a[PIECE];
                tmem_ld_n<PIECE>(lane_addr + c0, a);
                float4 hv[PIECE / 4];
#pragma unroll
                for (int i = 0; i < PIECE / 4; ++i)
                    hv[i] = c0 == cg * CW ? hv0[i] : *reinterpret_cast<const float4*>(p.h + hin_base + (int64_t)(c0 / 4 + i) * hin_stride);
                float v[PIECE];
#pragma unroll
                for (int i = 0; i < PIECE / 4; ++i) {
                    const float4 bb = *reinterpret_cast<const float4*>(v_bo + c0 + 4 * i);
                    v[4 * i] = hv[i].x + bb.x; v[4 * i + 1] = hv[i].y + bb.y; v[4 * i + 2] = hv[i].z + bb.z; v[4 * i + 3] = hv[i].w + bb.w;
                }
                ptx::tmem_ld_wait();
#pragma unroll
                for (int i = 0; i < PIECE; ++i) { v[i] += __uint_as_float(a[i]); a[i] = __float_as_uint(v[i]); }
                tmem_st_n<PIECE>(lane_addr + c0, a);
                stats_piece<PIECE>(v, sn, smean, sm2);
            }
            float mu, rstd;
            row_stats(sn, smean, sm2, mu, rstd);
            ptx::tmem_st_wait();
#pragma unroll
            for (int c0 = cg * CW; c0 < (cg + 1) * CW; c0 += PIECE) {
                uint32_t a[PIECE];
                tmem_ld_n<PIECE>(lane_addr + c0, a);
                ptx::tmem_ld_wait();
                const int kb = c0 >> 6;
#pragma unroll
                for (int j = 0; j < PIECE / 8; ++j) {
                    uint32_t hi[4], lo[4];
#pragma unroll
                    for (int i = 0; i < 4; ++i) {
                        const int col = c0 + 8 * j + 2 * i;
                        const float2 gg = *reinterpret_cast<const float2*>(v_g2 + col), bb = *reinterpret_cast<const float2*>(v_b2ln + col);
                        const float2 y = make_float2((__uint_as_float(a[8 * j + 2 * i]) - mu) * rstd * gg.x + bb.x,
                                                     (__uint_as_float(a[8 * j + 2 * i + 1]) - mu) * rstd * gg.y + bb.y);
                        split_bf16x2(y, hi[i], lo[i]);
                    }
                    const int ch = ((c0 & 63) >> 3) + j;                 // 16-byte chunk of the 128-byte swizzled row
                    const uint32_t off = kb * POST_SLOT + r * 128 + ((ch ^ (r & 7)) << 4);
                    asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(sA + off), "r"(hi[0]), "r"(hi[1]), "r"(hi[2]), "r"(hi[3]) : "memory");
                    asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(sA + KB * POST_SLOT + off), "r"(lo[0]), "r"(lo[1]), "r"(lo[2]), "r"(lo[3]) : "memory");
                    if (p.dbg_u2 && row_ok)
                        *reinterpret_cast<uint4*>(p.dbg_u2 + (int64_t)row * D + c0 + 8 * j) = make_uint4(hi[0], hi[1], hi[2], hi[3]);
                }
            }
            ptx::fence_proxy_async();                     // generic-proxy writes of u2 -> visible to the MMA's async proxy
            ptx::tc_fence_before();
            __syncwarp();
            if (lane == 0) ptx::mbar_arrive(bar_u2);

            // ---------------- FFN hidden chunks: g = act(S + b1) written back over S as packed bf16 (hi | lo)
            for (int c = 0; c < NC; ++c) {
                const int bsel = c & 1;
                ptx::mbar_wait(bar_s_full + 8 * bsel, (ph_s >> bsel) & 1);
                ph_s ^= 1u << bsel;
                ptx::tc_fence_after();
                const uint32_t s_addr = lane_addr + 256 + 128 * bsel + 32 * cg;
                uint32_t sv[32];
                ptx::tmem_ld32(s_addr, sv);
                ptx::tmem_ld_wait();
                const float* bp = v_b1 + c * POST_CH + 32 * cg;
                uint32_t hi[16], lo[16];
#pragma unroll
                for (int i = 0; i < 8; ++i) {
                    const float4 bb = *reinterpret_cast<const float4*>(bp + 4 * i);      // broadcast LDS.128
                    float2 x0 = ptx::fadd2(make_float2(__uint_as_float(sv[4 * i]), __uint_as_float(sv[4 * i + 1])), make_float2(bb.x, bb.y));
                    float2 x1 = ptx::fadd2(make_float2(__uint_as_float(sv[4 * i + 2]), __uint_as_float(sv[4 * i + 3])), make_float2(bb.z, bb.w));
                    split_bf16x2(act2<ACT>(x0), hi[2 * i], lo[2 * i]);
                    split_bf16x2(act2<ACT>(x1), hi[2 * i + 1], lo[2 * i + 1]);
                }
                ptx::tmem_st16(s_addr, hi);
                ptx::tmem_st16(s_addr + 16, lo);
                if (p.dbg_g && row_ok) {
                    uint4* gp = reinterpret_cast<uint4*>(p.dbg_g + (int64_t)row * p.dff + c * POST_CH + 32 * cg);
#pragma unroll
                    for (int i = 0; i < 4; ++i) gp[i] = make_uint4(hi[4 * i], hi[4 * i + 1], hi[4 * i + 2], hi[4 * i + 3]);
                }
                ptx::tmem_st_wait();
                ptx::tc_fence_before();
                __syncwarp();
                if (lane == 0) ptx::mbar_arrive(bar_g + 8 * bsel);
            }

            // ---------------- epilogue of FFN2: h2 = acc + b2 -> h (fp32); u' = LN_next(h2) -> bf16 hi (+ lo)
            ptx::mbar_wait(bar_acc_final, it & 1);
            ptx::tc_fence_after();
            sn = 0.f; smean = 0.f; sm2 = 0.f;
#pragma unroll
            for (int c0 = cg * CW; c0 < (cg + 1) * CW; c0 += PIECE) {
                uint32_t a[PIECE];
                tmem_ld_n<PIECE>(lane_addr + c0, a);
                ptx::tmem_ld_wait();
                float v[PIECE];
#pragma unroll
                for (int i = 0; i < PIECE / 4; ++i) {
                    const float4 bb = *reinterpret_cast<const float4*>(v_b2 + c0 + 4 * i);
                    v[4 * i] = __uint_as_float(a[4 * i]) + bb.x; v[4 * i + 1] = __uint_as_float(a[4 * i + 1]) + bb.y;
                    v[4 * i + 2] = __uint_as_float(a[4 * i + 2]) + bb.z; v[4 * i + 3] = __uint_as_float(a[4 * i + 3]) + bb.w;
                }
                if (row_ok) {
#pragma unroll
                    for (int i = 0; i < PIECE / 4; ++i)
                        *reinterpret_cast<float4*>(p.h + hout_base + (int64_t)(c0 / 4 + i) * hout_stride) = make_float4(v[4 * i], v[4 * i + 1], v[4 * i + 2], v[4 * i + 3]);
                }
                stats_piece<PIECE>(v, sn, smean, sm2);
            }
            row_stats(sn, smean, sm2, mu, rstd);
            if (!p.next_ln) { mu = 0.0f; rstd = 1.0f; }
#pragma unroll
            for (int c0 = cg * CW; c0 < (cg + 1) * CW; c0 += PIECE) {
                uint32_t a[PIECE];
                tmem_ld_n<PIECE>(lane_addr + c0, a);
                ptx::tmem_ld_wait();
                uint32_t hi[PIECE / 2], lo[PIECE / 2], f8[PIECE / 4];
#pragma unroll
                for (int i = 0; i < PIECE / 2; ++i) {
                    const int col = c0 + 2 * i;
                    const float2 b2v = *reinterpret_cast<const float2*>(v_b2 + col);
                    const float2 gg = *reinterpret_cast<const float2*>(v_gn + col), bb = *reinterpret_cast<const float2*>(v_bn + col);
                    const float2 y = make_float2((__uint_as_float(a[2 * i]) + b2v.x - mu) * rstd * gg.x + bb.x,
                                                 (__uint_as_float(a[2 * i + 1]) + b2v.y - mu) * rstd * gg.y + bb.y);
                    split_bf16x2(y, hi[i], lo[i]);
                    if (p.u_out_f8) {                       // (lo[] is free to carry the e4m3 pairs when there is no lo output)
                        const uint32_t q = __nv_cvt_float2_to_fp8x2(make_float2(y.x * p.f8_scale, y.y * p.f8_scale), __NV_SATFINITE, __NV_E4M3);
                        if (i & 1) f8[i >> 1] |= q << 16; else f8[i >> 1] = q;
                    }
                }
                if (row_ok && p.u_out_f8) {
#pragma unroll
                    for (int j = 0; j < PIECE / 16; ++j)
                        *reinterpret_cast<uint4*>(p.u_out_f8 + (int64_t)row * D + c0 + 16 * j) = make_uint4(f8[4 * j], f8[4 * j + 1], f8[4 * j + 2], f8[4 * j + 3]);
                }
                if (row_ok) {                             // 32-byte stores: a full sector per lane
#pragma unroll
                    for (int j = 0; j < PIECE / 16; ++j) {
                        st_global_v8(p.u_out + (int64_t)row * D + c0 + 16 * j, &hi[8 * j]);
                        if (p.u_out_lo) st_global_v8(p.u_out_lo + (int64_t)row * D + c0 + 16 * j, &lo[8 * j]);
                    }
                }
            }
            ptx::tc_fence_before();
            __syncwarp();
            if (lane == 0) ptx::mbar_arrive(bar_acc_free);
        }
    }
    ptx::tc_fence_before();
    __syncthreads();
    if (warp == 1) ptx::tmem_dealloc(tmem_base, 512);
}

// ------------------------------------------------------------------------------------------------ launch
bool tc_post_supported(int d, int dff) {
    if (d != 64 && d != 128 && d != 256) return false;
    if (dff < POST_CH || dff % POST_CH) return false;
    const int smem = d == 64 ? PostCfg<64>::smem_bytes(dff) : d == 128 ? PostCfg<128>::smem_bytes(dff) : PostCfg<256>::smem_bytes(dff);
    return smem + 512 <= 232448;                          // 227 KB per CTA, static shared memory included
}

template <int D, int ACT>
static int tc_post_launch_t(TcContext* c, const PostArgs& a, cudaStream_t st) {
    using Cfg = PostCfg<D>;
    CUtensorMap tmO, tmOlo, tmWo, tmW1, tmW2;
    const int G = a.n_groups;
    if (tc_tensor_map(c, &tmO, a.o, D, a.M, D, 64, POST_BM)) return -1;
    if (tc_tensor_map(c, &tmOlo, a.o_lo, D, a.M, D, 64, POST_BM)) return -1;
    if (tc_tensor_map(c, &tmWo, a.Wo, D, (uint64_t)G * D, D, 64, Cfg::NB)) return -1;
    if (tc_tensor_map(c, &tmW1, a.W1, D, (uint64_t)G * a.dff, D, 64, POST_CH)) return -1;
    if (tc_tensor_map(c, &tmW2, a.W2, a.dff, (uint64_t)G * D, a.dff, 64, Cfg::NB)) return -1;
    auto kern = k_tc_post<D, ACT>;
    const int smem = Cfg::smem_bytes(a.dff);
    if (tc_set_smem_attr(c, (const void*)kern, 232448 - 1024)) return -1;   // upper bound once per device; dff varies per model
    PostParams p;
    p.M = a.M; p.dff = a.dff; p.group_rows = a.group_rows > 0 ? a.group_rows : 0x7fffff80; p.nc_dev = a.nc_dev;
    p.bo = a.bo; p.ln2g = a.ln2g; p.ln2b = a.ln2b; p.b1 = a.b1; p.b2 = a.b2; p.lnng = a.lnng; p.lnnb = a.lnnb;
    p.eps = a.eps; p.h = a.h; p.h_in_tiled = a.h_in_tiled; p.h_out_tiled = a.h_out_tiled; p.u_out = a.u_out; p.u_out_lo = a.u_out_lo; p.next_ln = a.next_ln;
    p.dbg_u2 = a.dbg_u2; p.dbg_g = a.dbg_g; p.u_out_f8 = a.u_out_f8; p.f8_scale = a.f8_scale;
    const int n_tiles = (a.M + POST_BM - 1) / POST_BM;
    const int grid = n_tiles < c->num_sms ? n_tiles : c->num_sms;
    tc_launch(kern, dim3(grid), dim3(POST_THREADS), smem, st, c->pdl, tmO, tmOlo, tmWo, tmW1, tmW2, p);
    return 0;
}

int tc_post_launch(TcContext* c, const PostArgs& a, cudaStream_t st) {
    if (!tc_post_supported(a.d, a.dff) || !a.o || !a.o_lo || !a.u_out || (a.act != ACT_GELU && a.act != ACT_RELU)) {
        snprintf(c->err, sizeof c->err, "tc_post: unsupported shape d=%d dff=%d act=%d", a.d, a.dff, a.act);
        return -1;
    }
#define POST_CASE(DD) \
    if (a.d == DD) return a.act == ACT_GELU ? tc_post_launch_t<DD, ACT_GELU>(c, a, st) : tc_post_launch_t<DD, ACT_RELU>(c, a, st);
    POST_CASE(64) POST_CASE(128) POST_CASE(256)
#undef POST_CASE
    return -1;
}

}  // namespace mlpf
