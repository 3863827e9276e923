// tc_attn.cuh -- varlen, key-padding-masked flash-attention forward on tcgen05 / TMEM / TMA (sm_100a).
// Step a4 of DESIGN.md:  per event, per head  O = softmax(Q K^T / sqrt(hd) + mask) V   (Eq. 4),
// computed with the FlashAttention recurrence (running max / running sum over key tiles, L154) so the
// n x n weight matrix never leaves the SM.  Keys outside the event or with key_valid == 0 get weight
// exactly 0 (reading A2); a query with no valid key gets O = 0 (A15).
//
// One CTA = one head x two consecutive 128-row query tiles (a, b) of one event, sharing every K / V^T tile.
//   warp 0      TMA producer: Q_a, Q_b once; then (K_j, V_j), each [128 keys x hd] row-major, into a ring.
//               Q, K, V are column blocks of one row-major [N, 3d] buffer, so an event may start at any row
//               (TMA needs 16-byte alignment only along the innermost, head-dim, coordinate).
//   warp 1      MMA issuer:   S_t = Q_t K_j^T  (M=128, N=128, K=hd)  -> TMEM (fp32);
//                             O_t(j) = P_t V_j (A = P_t read from TMEM, B = V_j as an MN-major operand,
//                             K=128, N=hd) -> TMEM, fresh each tile.
//   warps 2-5   softmax warpgroup of tile a, warps 6-9 of tile b: one query row per thread:
//               S -> (mask) -> running max -> exp2 -> bf16 P written back over S's columns in TMEM;
//               then acc = acc * corr + O_t(j-1) in registers (no read-modify-write of O in TMEM).
// The two warpgroups run half a period apart (S_t(j+1) is issued right after P_t(j) V_j), so one of
// them is exponentiating while the other waits for the tensor pipe.
// TMEM columns: S_a [0,128) S_b [128,256) (P_t aliases the first 64 columns of S_t), O_t[buf] at 256 + (2t+buf) hd.
#include "tc_api.h"
#include "ptx.cuh"

namespace mlpf {

constexpr int ATT_THREADS = 320;
constexpr int ATT_BQ = 128, ATT_BK = 128;

template <int HD>
struct AttnCfg {
    static constexpr int Q_BYTES = ATT_BQ * HD * 2;
    static constexpr int K_BYTES = ATT_BK * HD * 2;
    static constexpr int V_BYTES = HD * ATT_BK * 2;
    static constexpr int STAGE_BYTES = K_BYTES + V_BYTES;
    static constexpr int STAGES = HD == 64 ? 4 : 6;
    static constexpr int SMEM_BYTES = 2 * Q_BYTES + STAGES * STAGE_BYTES + 1024;
    static constexpr int SW = HD * 2;                       // swizzle width of Q / K rows in bytes
};

struct AttnParams {
    const int* key_valid;      // [N] or null
    const int* offsets;        // [E+1]
    const int2* pairs;         // (event, pair index)
    int n_pairs, H, d;
    bf16* O; bf16* O_lo;
    float scale_log2;          // log2(e) / sqrt(hd)
};

template <int HD>
__global__ void __launch_bounds__(ATT_THREADS, 1)
k_tc_attn(const __grid_constant__ CUtensorMap tmQKV, AttnParams prm) {
    using Cfg = AttnCfg<HD>;
    constexpr int ST = Cfg::STAGES;
    extern __shared__ uint8_t smem_raw[];
    __shared__ uint64_t bars[1 + 2 * ST + 6];
    __shared__ uint32_t tmem_base_slot;

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int item = blockIdx.x / prm.H, head = blockIdx.x % prm.H;
    const int2 pr = prm.pairs[item];
    const int ev0 = prm.offsets[pr.x], ev1 = prm.offsets[pr.x + 1];
    const int q0a = ev0 + pr.y * 2 * ATT_BQ, q0b = q0a + ATT_BQ;
    const bool has_b = q0b < ev1;
    const int nkv = (ev1 - ev0 + ATT_BK - 1) / ATT_BK;

    const uint32_t smem_base = (ptx::smem_u32(smem_raw) + 1023u) & ~1023u;
    const uint32_t sQ = smem_base;                                  // Q_a, Q_b
    const uint32_t sKV = smem_base + 2 * Cfg::Q_BYTES;
    const uint32_t bar_q = ptx::smem_u32(&bars[0]);
    const uint32_t bar_kv_full = ptx::smem_u32(&bars[1]);
    const uint32_t bar_kv_empty = ptx::smem_u32(&bars[1 + ST]);
    const uint32_t bar_s = ptx::smem_u32(&bars[1 + 2 * ST]);        // [t]
    const uint32_t bar_p = ptx::smem_u32(&bars[1 + 2 * ST + 2]);    // [t]
    const uint32_t bar_o = ptx::smem_u32(&bars[1 + 2 * ST + 4]);    // [t]

    if (warp == 0 && lane == 0) {
        ptx::mbar_init(bar_q, 1);
        for (int s = 0; s < ST; ++s) { ptx::mbar_init(bar_kv_full + 8 * s, 1); ptx::mbar_init(bar_kv_empty + 8 * s, 1); }
        for (int t = 0; t < 2; ++t) {
            ptx::mbar_init(bar_s + 8 * t, 1);
            ptx::mbar_init(bar_p + 8 * t, 4);                        // one arrival per softmax warp
            ptx::mbar_init(bar_o + 8 * t, 1);
        }
        ptx::fence_barrier_init();
        ptx::tma_prefetch_desc(&tmQKV);
    }
    if (warp == 1) {
        ptx::tmem_alloc(ptx::smem_u32(&tmem_base_slot), 512);
        ptx::tmem_relinquish();
    }
    ptx::tc_fence_before();
    __syncthreads();
    ptx::tc_fence_after();
    const uint32_t tmem_base = tmem_base_slot;

    if (warp == 0) {
        // ------------------------------------------------------------ TMA producer
        if (lane == 0) {
            ptx::mbar_expect_tx(bar_q, Cfg::Q_BYTES * (has_b ? 2 : 1));
            ptx::tma_load_2d(sQ, &tmQKV, bar_q, head * HD, q0a);
            if (has_b) ptx::tma_load_2d(sQ + Cfg::Q_BYTES, &tmQKV, bar_q, head * HD, q0b);
        }
        for (int j = 0; j < nkv; ++j) {
            const int s = j % ST;
            ptx::mbar_wait(bar_kv_empty + 8 * s, ((j / ST) & 1) ^ 1);
            if (lane == 0) {
                const uint32_t st = sKV + s * Cfg::STAGE_BYTES;
                const int k0 = ev0 + j * ATT_BK;
                ptx::mbar_expect_tx(bar_kv_full + 8 * s, Cfg::STAGE_BYTES);
                ptx::tma_load_2d(st, &tmQKV, bar_kv_full + 8 * s, prm.d + head * HD, k0);
                ptx::tma_load_2d(st + Cfg::K_BYTES, &tmQKV, bar_kv_full + 8 * s, 2 * prm.d + head * HD, k0);
            }
            __syncwarp();
        }
    } else if (warp == 1) {
        // ------------------------------------------------------------ MMA issuer
        constexpr uint32_t idesc_s = ptx::umma_idesc_bf16(128, ATT_BK);
        constexpr uint32_t idesc_o = ptx::umma_idesc_bf16(128, HD) | ptx::UMMA_B_MN_MAJOR;
        auto issue_s = [&](int t, int j) {          // S_t = Q_t K_j^T
            const uint32_t kb = sKV + (j % ST) * Cfg::STAGE_BYTES;
            const uint32_t qb = sQ + t * Cfg::Q_BYTES;
#pragma unroll
            for (int k = 0; k < HD / 16; ++k)
                ptx::mma_ss(tmem_base + t * 128, ptx::umma_desc_kmajor(qb + k * 32, Cfg::SW),
                            ptx::umma_desc_kmajor(kb + k * 32, Cfg::SW), idesc_s, k != 0);
            ptx::mma_commit(bar_s + 8 * t);
        };
        auto issue_o = [&](int t, int j) {          // O_t(j) = P_t V_j
            const uint32_t vb = sKV + (j % ST) * Cfg::STAGE_BYTES + Cfg::K_BYTES;
            const uint32_t o_col = 256 + (2 * t + (j & 1)) * HD;
#pragma unroll
            for (int k = 0; k < ATT_BK / 16; ++k)
                ptx::mma_ts(tmem_base + o_col, tmem_base + t * 128 + k * 8,
                            ptx::umma_desc_mnmajor(vb + k * 16 * Cfg::SW, Cfg::SW), idesc_o, k != 0);
            ptx::mma_commit(bar_o + 8 * t);
        };
        ptx::mbar_wait(bar_q, 0);
        ptx::mbar_wait(bar_kv_full, 0);
        ptx::tc_fence_after();
        if (lane == 0) { issue_s(0, 0); if (has_b) issue_s(1, 0); }
        __syncwarp();
        for (int j = 0; j < nkv; ++j) {
            const uint32_t par = j & 1;
            const bool more = j + 1 < nkv;
            if (more) ptx::mbar_wait(bar_kv_full + 8 * ((j + 1) % ST), ((j + 1) / ST) & 1);
            ptx::mbar_wait(bar_p, par);                           // P_a(j) is in TMEM
            ptx::tc_fence_after();
            if (lane == 0) {
                issue_o(0, j);
                if (!has_b) ptx::mma_commit(bar_kv_empty + 8 * (j % ST));
                if (more) issue_s(0, j + 1);
            }
            __syncwarp();
            if (has_b) {
                ptx::mbar_wait(bar_p + 8, par);
                ptx::tc_fence_after();
                if (lane == 0) {
                    issue_o(1, j);
                    ptx::mma_commit(bar_kv_empty + 8 * (j % ST));
                    if (more) issue_s(1, j + 1);
                }
                __syncwarp();
            }
        }
    } else {
        // ------------------------------------------------------------ softmax warpgroups
        const int t = (warp - 2) >> 2;                 // 0: tile a, 1: tile b
        const int q = warp & 3;                        // TMEM lane quarter this warp may access
        const int row_in_tile = q * 32 + lane;
        const int qrow = (t == 0 ? q0a : q0b) + row_in_tile;
        if (t == 0 || has_b) {
            const uint32_t lane_addr = tmem_base + ((uint32_t)(q * 32) << 16);
            const uint32_t s_addr = lane_addr + t * 128;
            const float c = prm.scale_log2;
            float acc[HD];
#pragma unroll
            for (int i = 0; i < HD; ++i) acc[i] = 0.0f;
            float m_run = -INFINITY, l_run = 0.0f, corr_prev = 0.0f;
            for (int j = 0; j < nkv; ++j) {
                // key mask of this tile: 4 x 32 bits, computed redundantly per warp (no cross-warp sync)
                const int k0 = ev0 + j * ATT_BK;
                uint32_t mask[4];
#pragma unroll
                for (int w = 0; w < 4; ++w) {
                    const int key = k0 + w * 32 + lane;
                    bool ok = key < ev1;
                    if (ok && prm.key_valid) ok = prm.key_valid[key] != 0;
                    mask[w] = __ballot_sync(0xffffffffu, ok);
                }
                const bool full = (mask[0] & mask[1] & mask[2] & mask[3]) == 0xffffffffu;
                ptx::mbar_wait(bar_s + 8 * t, j & 1);
                ptx::tc_fence_after();
                // pass 1: row max
                float mx = -INFINITY;
#pragma unroll
                for (int w = 0; w < 4; ++w) {
                    uint32_t r[32];
                    ptx::tmem_ld32(s_addr + w * 32, r);
                    ptx::tmem_ld_wait();
                    if (full) {
#pragma unroll
                        for (int i = 0; i < 32; ++i) mx = fmaxf(mx, __uint_as_float(r[i]));
                    } else {
#pragma unroll
                        for (int i = 0; i < 32; ++i)
                            mx = fmaxf(mx, (mask[w] >> i) & 1u ? __uint_as_float(r[i]) : -INFINITY);
                    }
                }
                const float m_new = fmaxf(m_run, mx);
                const float m_use = (m_new == -INFINITY) ? 0.0f : m_new;
                const float corr = ptx::fast_exp2((m_run - m_use) * c);          // m_run = -inf -> 0
                const float neg_mc = -m_use * c;
                float rsum = 0.0f;
                // pass 2: P = exp2(S c - m c) as bf16 pairs, written over S's first 64 columns
#pragma unroll
                for (int w = 0; w < 4; ++w) {
                    uint32_t r[32];
                    ptx::tmem_ld32(s_addr + w * 32, r);
                    ptx::tmem_ld_wait();
                    uint32_t pk[16];
#pragma unroll
                    for (int i = 0; i < 16; ++i) {
                        float p0 = ptx::fast_exp2(fmaf(__uint_as_float(r[2 * i]), c, neg_mc));
                        float p1 = ptx::fast_exp2(fmaf(__uint_as_float(r[2 * i + 1]), c, neg_mc));
                        if (!full) {
                            p0 = (mask[w] >> (2 * i)) & 1u ? p0 : 0.0f;
                            p1 = (mask[w] >> (2 * i + 1)) & 1u ? p1 : 0.0f;
                        }
                        rsum += p0 + p1;
                        __nv_bfloat162 b2 = __floats2bfloat162_rn(p0, p1);
                        pk[i] = *reinterpret_cast<uint32_t*>(&b2);
                    }
                    ptx::tmem_st16(s_addr + w * 16, pk);
                }
                ptx::tmem_st_wait();
                ptx::tc_fence_before();
                // O_t(j-1) was issued a whole softmax period ago: this wait does not stall, but it must come
                // BEFORE P_t(j) is published -- afterwards O_t(j) could complete too and the barrier would be two
                // phases ahead of this waiter (parity aliasing).
                if (j > 0) ptx::mbar_wait(bar_o + 8 * t, (j - 1) & 1);
                __syncwarp();
                if (lane == 0) ptx::mbar_arrive(bar_p + 8 * t);
                l_run = l_run * corr + rsum;
                m_run = m_new;
                // fold the previous tile's P V into the register accumulator
                if (j > 0) {
                    ptx::tc_fence_after();
                    const uint32_t o_addr = lane_addr + 256 + (2 * t + ((j - 1) & 1)) * HD;
#pragma unroll
                    for (int w = 0; w < HD / 16; ++w) {
                        uint32_t r[16];
                        ptx::tmem_ld16(o_addr + w * 16, r);
                        ptx::tmem_ld_wait();
#pragma unroll
                        for (int i = 0; i < 16; ++i) acc[w * 16 + i] = fmaf(acc[w * 16 + i], corr_prev, __uint_as_float(r[i]));
                    }
                }
                corr_prev = corr;
            }
            // last tile's P V
            {
                const int j = nkv - 1;
                ptx::mbar_wait(bar_o + 8 * t, j & 1);
                ptx::tc_fence_after();
                const uint32_t o_addr = lane_addr + 256 + (2 * t + (j & 1)) * HD;
#pragma unroll
                for (int w = 0; w < HD / 16; ++w) {
                    uint32_t r[16];
                    ptx::tmem_ld16(o_addr + w * 16, r);
                    ptx::tmem_ld_wait();
#pragma unroll
                    for (int i = 0; i < 16; ++i) acc[w * 16 + i] = fmaf(acc[w * 16 + i], corr_prev, __uint_as_float(r[i]));
                }
            }
            if (qrow < ev1) {
                const float inv = l_run > 0.0f ? 1.0f / l_run : 0.0f;
                uint32_t hi[HD / 2], lo[HD / 2];
#pragma unroll
                for (int i = 0; i < HD / 2; ++i) {
                    const float y0 = acc[2 * i] * inv, y1 = acc[2 * i + 1] * inv;
                    __nv_bfloat162 h2 = __floats2bfloat162_rn(y0, y1);
                    hi[i] = *reinterpret_cast<uint32_t*>(&h2);
                    __nv_bfloat162 l2 = __floats2bfloat162_rn(y0 - __low2float(h2), y1 - __high2float(h2));
                    lo[i] = *reinterpret_cast<uint32_t*>(&l2);
                }
                uint4* op = reinterpret_cast<uint4*>(prm.O + (int64_t)qrow * prm.d + head * HD);
#pragma unroll
                for (int i = 0; i < HD / 8; ++i) op[i] = make_uint4(hi[4 * i], hi[4 * i + 1], hi[4 * i + 2], hi[4 * i + 3]);
                if (prm.O_lo) {
                    uint4* lp = reinterpret_cast<uint4*>(prm.O_lo + (int64_t)qrow * prm.d + head * HD);
#pragma unroll
                    for (int i = 0; i < HD / 8; ++i) lp[i] = make_uint4(lo[4 * i], lo[4 * i + 1], lo[4 * i + 2], lo[4 * i + 3]);
                }
            }
        }
    }
    ptx::tc_fence_before();
    __syncthreads();
    if (warp == 1) ptx::tmem_dealloc(tmem_base, 512);
}

template <int HD>
static int tc_attn_launch_hd(TcContext* c, const bf16* QKV, int64_t N, const AttnParams& prm,
                             cudaStream_t st) {
    using Cfg = AttnCfg<HD>;
    CUtensorMap tmQKV;
    if (tc_tensor_map(c, &tmQKV, QKV, 3 * prm.d, N, 3 * prm.d, HD, ATT_BQ)) return -1;
    auto kern = k_tc_attn<HD>;
    static bool attr_set = false;
    if (!attr_set) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, Cfg::SMEM_BYTES);
        if (e != cudaSuccess) { snprintf(c->err, sizeof c->err, "cudaFuncSetAttribute: %s", cudaGetErrorString(e)); return -1; }
        attr_set = true;
    }
    kern<<<prm.n_pairs * prm.H, ATT_THREADS, Cfg::SMEM_BYTES, st>>>(tmQKV, prm);
    return 0;
}

int tc_attn_launch(TcContext* c, const bf16* QKV, int64_t N, const int* key_valid,
                          const int* offsets, const int2* pairs, int n_pairs, int d, int H, bf16* O, bf16* O_lo,
                          cudaStream_t st) {
    const int hd = d / H;
    AttnParams prm;
    prm.key_valid = key_valid; prm.offsets = offsets; prm.pairs = pairs; prm.n_pairs = n_pairs; prm.H = H; prm.d = d;
    prm.O = O; prm.O_lo = O_lo;
    prm.scale_log2 = 1.4426950408889634f / sqrtf((float)hd);
    switch (hd) {
        case 16: return tc_attn_launch_hd<16>(c, QKV, N, prm, st);
        case 32: return tc_attn_launch_hd<32>(c, QKV, N, prm, st);
        case 64: return tc_attn_launch_hd<64>(c, QKV, N, prm, st);
    }
    snprintf(c->err, sizeof c->err, "tc_attn: head_dim %d unsupported", hd);
    return -1;
}

}  // namespace mlpf
