// tc_attn.cu -- varlen, key-padding-masked flash-attention forward on tcgen05 / TMEM / TMA (sm_100a).
// Step a4 of DESIGN.md:  per event, per head  O = softmax(Q K^T / sqrt(hd) + mask) V   (Eq. 4),
// computed with the FlashAttention recurrence (running max / running sum over key tiles, L154) so the
// n x n weight matrix never leaves the SM.  Keys outside the event or with key_valid == 0 get weight
// exactly 0 (reading A2); a query with no valid key gets O = 0 (A15).
//
// One CTA = one head x NT consecutive 128-row query tiles of one event (NT = 3 at hd <= 32, 2 at hd = 64),
// sharing every K / V tile.  Key tiles are 64 keys wide and S is DOUBLE-BUFFERED in TMEM, so the tensor pipe
// computes S_t(j+1) while the softmax warps work on S_t(j): the MMA chain (issue + hand-off latency) is off the
// softmax warps' critical path.  At hd = 32 the exponentials (MUFU, 16/clk/SM) are the binding unit; one softmax
// warp's serial chain per tile (TMEM load, max, exp, TMEM store, fold) is about twice its MUFU time, so three
// warps per SM sub-partition (NT = 3) are what keeps the MUFU pipe busy.
//   warps 0 .. 4NT-1   softmax warpgroups, one per query tile: one query row per thread, the tile's 64 scores in
//               registers:  S -> (mask) -> max -> P = 2^((S - m_ref) c) as bf16 written back over S's TMEM columns.
//               m_ref is a stale reference maximum (lazy rescaling): O_t and the row sums accumulate in TMEM over
//               all key tiles and are rescaled in place only when m_ref moves (a few times per row).
//   warp 4NT    TMA producer: Q tiles once; then stages of (K, V), each [128 keys x hd] row-major (two key tiles
//               per stage).  Q, K, V are column blocks of one row-major [N, 3d] buffer, so an event may start at
//               any row (TMA needs 16-byte alignment only along the innermost, head-dim, coordinate).
//   warps 4NT+1 .. 4NT+NT   MMA issuers, one per query tile:  S_t(j) = Q_t K_j^T  (M=128, N=64, K=hd) -> S buffer
//               j&1;  O_t += P_t(j) V_j (A = P read from TMEM, B = V_j as an MN-major operand, K=64, N=hd) and
//               l_t += P_t(j) 1 (N = 8, a tile of ones as B): the softmax denominators.
//               All 32 lanes run the issue code with warp-uniform operands (one lane elected inside the wrappers).
// setmaxnreg moves the producer warpgroup's registers to the softmax warpgroups.
// TMEM columns: S_t[b] at 128 t + 64 b (P_t[b] aliases its first 32 columns); O_t | l_t at 128 NT + (hd + 8) t.
#include "tc_api.h"
#include "ptx.cuh"
#include <type_traits>

namespace mlpf {

constexpr int ATT_BQ = 128, ATT_BK = 64, ATT_SK = 128;  // query tile, key tile, keys per TMA stage

template <int HD>
struct AttnCfg {
    static constexpr int NT = HD <= 32 ? 3 : 2;             // query tiles per CTA
    static constexpr int THREADS = (NT + 1) * 128;
    static constexpr int WARP_TMA = 4 * NT, WARP_MMA = 4 * NT + 1;
    static constexpr int SOFTMAX_REGS = NT == 3 ? 152 : 232, PRODUCER_REGS = 40;
    static constexpr int Q_BYTES = ATT_BQ * HD * 2;
    static constexpr int K_BYTES = ATT_SK * HD * 2;
    static constexpr int V_BYTES = ATT_SK * HD * 2;
    static constexpr int STAGE_BYTES = K_BYTES + V_BYTES;
    static constexpr int STAGES = HD == 64 ? 4 : 6;
    static constexpr int ONES_BYTES = 1024;                 // bf16 1.0: B operand of the row-sum MMA (any layout reads ones)
    static constexpr int OW = HD + 8;                       // TMEM columns per query tile: O (hd) + row sums (8 equal columns)
    static constexpr int SMEM_BYTES = NT * Q_BYTES + STAGES * STAGE_BYTES + ONES_BYTES + 1024;
    static constexpr int SW = HD * 2;                       // swizzle width of Q / K / V rows in bytes
    static constexpr int O_COL0 = 128 * NT;
    static_assert(O_COL0 + NT * OW <= 512, "TMEM budget");
};

int tc_attn_rows_per_cta(int hd) { return (hd <= 32 ? 3 : 2) * ATT_BQ; }

struct AttnParams {
    const uint32_t* valid_bits; // one bit per row, 32 rows per word (3 readable words past the last row's), or null
    const int* n_valid;        // [E] valid rows per event, or null: events without pad rows skip the key_valid loads
    const int* offsets;        // [E+1]
    const int2* items;         // (event, index of the group of NT query tiles)
    int n_items, H, d;
    bf16* O; bf16* O_lo;
    float scale_log2;          // log2(e) / sqrt(hd)
};

// 32 scores of one row (registers r[0..31]) -> max, as four independent chains (a single chain of 32 dependent
// FMNMX costs ~200 cycles of latency that nothing else in the warp can hide)
template <bool FULL>
__device__ __forceinline__ float max32(const uint32_t* r, uint32_t mask, float mx) {
    float m[4] = {mx, -INFINITY, -INFINITY, -INFINITY};
#pragma unroll
    for (int i = 0; i < 32; ++i) {
        const float v = __uint_as_float(r[i]);
        m[i & 3] = fmaxf(m[i & 3], FULL ? v : ((mask >> i) & 1u ? v : -INFINITY));
    }
    return fmaxf(fmaxf(m[0], m[1]), fmaxf(m[2], m[3]));
}
// 2^x for a pair, x <= 0, on the FMA / ALU pipes instead of the MUFU (Cody-Waite split + degree-3 polynomial):
//   x = n + f, n = round(x) taken from the mantissa of x + 1.5 * 2^23, f in [-0.5, 0.5];
//   2^f ~ 1 + f (c1 + f (c2 + f c3))  (max relative error 1.0e-4, 40x below the bf16 rounding of P);
//   2^n goes into the exponent field with one integer multiply-add.
// The MUFU does 16 ex2 per clock and SM and is the binding unit of this kernel at hd = 32 (one ex2 per 128 tensor
// FLOPs); every ATT_POLY_EVERY-th pair takes this path so that MUFU and FMA pipes finish together.
__device__ __forceinline__ float2 exp2_poly2(float2 x) {
    const float2 magic = make_float2(12582912.0f, 12582912.0f);
    x.x = fmaxf(x.x, -126.0f); x.y = fmaxf(x.y, -126.0f);
    const float2 xr = ptx::fadd2(x, magic);                                          // low mantissa bits = round(x)
    const float2 f = ptx::fadd2(x, ptx::fadd2(make_float2(12582912.0f, 12582912.0f), make_float2(-xr.x, -xr.y)));
    float2 p = ptx::ffma2(f, make_float2(0.0550089306f, 0.0550089306f), make_float2(0.2422109596f, 0.2422109596f));
    p = ptx::ffma2(p, f, make_float2(0.6932829272f, 0.6932829272f));
    p = ptx::ffma2(p, f, make_float2(1.0f, 1.0f));
    return make_float2(__int_as_float(__float_as_int(p.x) + (__float_as_int(xr.x) << 23)),
                       __int_as_float(__float_as_int(p.y) + (__float_as_int(xr.y) << 23)));
}
#ifndef ATT_POLY_POS
#define ATT_POLY_POS 0       // which pair of each group of ATT_POLY_EVERY (0 measured 1-2 % faster than the last)
#endif
#ifndef ATT_POLY_EVERY
#define ATT_POLY_EVERY 4     // measured on cfg3 (hd = 32, ms per layer): off 0.865, every 8th pair 0.845, 4th 0.825,
#endif                       // 3rd 0.846, 2nd 0.927 (with register spills in the loop it was a loss at every setting)


// p = 2^(s c - m c) for 32 scores -> 16 bf16 pairs (the row sums come from the tensor pipe: P x 1)
template <bool FULL, bool POLY>
__device__ __forceinline__ void exp32(const uint32_t* r, uint32_t mask, float c, float neg_mc, uint32_t (&pk)[16]) {
    const float2 c2 = make_float2(c, c), m2 = make_float2(neg_mc, neg_mc);
#pragma unroll
    for (int i = 0; i < 16; ++i) {
        const float2 x = ptx::ffma2(make_float2(__uint_as_float(r[2 * i]), __uint_as_float(r[2 * i + 1])), c2, m2);
        float2 p;
        if (POLY && ATT_POLY_EVERY > 0 && (i % (ATT_POLY_EVERY > 0 ? ATT_POLY_EVERY : 1)) == ATT_POLY_POS) p = exp2_poly2(x);
        else p = make_float2(ptx::fast_exp2(x.x), ptx::fast_exp2(x.y));
        if (!FULL) {
            p.x = (mask >> (2 * i)) & 1u ? p.x : 0.0f;
            p.y = (mask >> (2 * i + 1)) & 1u ? p.y : 0.0f;
        }
        __nv_bfloat162 b2 = __floats2bfloat162_rn(p.x, p.y);
        pk[i] = *reinterpret_cast<uint32_t*>(&b2);
    }
}

// One 64-key tile of one query row, scores already in registers s[0..63]:
// P = 2^((S - m_ref) c) as bf16, written over S's first 32 TMEM columns at s_addr.
// m_ref is a STALE reference maximum (lazy rescaling): it only moves when some row of the warp has a tile maximum
// more than ATT_RESCALE_LOG2 (in log2 units) above it, so P <= 2^8 and neither bf16 P nor the fp32 sums lose
// precision, while the accumulated O (in TMEM) has to be rescaled only a few times per row instead of every tile.
// Returns corr = 2^((m_ref_old - m_ref_new) c); `rescale` (warp-uniform) says whether m_ref moved.
constexpr float ATT_RESCALE_LOG2 = 8.0f;
template <bool FULL, bool POLY = true>
__device__ __forceinline__ float softmax_tile(const uint32_t (&s)[64], uint32_t s_addr, const uint32_t (&mask)[2], float c,
                                              float& m_ref, bool& rescale) {
    const float mx = fmaxf(max32<FULL>(&s[0], mask[0], -INFINITY), max32<FULL>(&s[32], mask[1], -INFINITY));
    const float m_new = fmaxf(m_ref, mx);
    // m_ref = -inf and a finite tile maximum: the difference is +inf and votes yes; all keys masked so far: nan -> no
    rescale = __any_sync(0xffffffffu, (m_new - m_ref) * c > ATT_RESCALE_LOG2);
    float corr = 1.0f;
    if (rescale) {
        const float m_use = (m_new == -INFINITY) ? 0.0f : m_new;
        corr = ptx::fast_exp2((m_ref - m_use) * c);              // m_ref = -inf -> 0
        m_ref = m_new;
    }
    const float neg_mc = (m_ref == -INFINITY) ? 0.0f : -m_ref * c;
#pragma unroll
    for (int w = 0; w < 2; ++w) {
        uint32_t pk[16];
        exp32<FULL, POLY>(&s[32 * w], mask[w], c, neg_mc, pk);
        ptx::tmem_st16(s_addr + 16 * w, pk);
    }
    return corr;
}

// Masked tile, hd = 64 variant: the scores of keys outside the event / of pad rows become -inf ONCE, so the max pass
// ignores them and 2^(-inf) gives the exact weight 0 on the MUFU (no polynomial path: it clamps its argument).  Two
// selects per score less than softmax_tile<false>.  Only instantiated at hd = 64: inside the hd <= 32 kernels the same
// code changed ptxas' schedule of the unmasked loop for the worse (cfg3 3 % slower: measured), there the padded
// configs matter less than the pad-free headline.
__device__ __forceinline__ float softmax_tile_mask_once(uint32_t (&s)[64], uint32_t s_addr, const uint32_t (&mask)[2], float c,
                                                        float& m_ref, bool& rescale) {
#pragma unroll
    for (int i = 0; i < 64; ++i) s[i] = (mask[i >> 5] >> (i & 31)) & 1u ? s[i] : 0xff800000u;
    return softmax_tile<true, false>(s, s_addr, mask, c, m_ref, rescale);
}

template <int HD>
__global__ void __launch_bounds__(AttnCfg<HD>::THREADS, 1)
k_tc_attn(const __grid_constant__ CUtensorMap tmQKV, AttnParams prm) {
    using Cfg = AttnCfg<HD>;
    constexpr int ST = Cfg::STAGES, NT = Cfg::NT;
    extern __shared__ uint8_t smem_raw[];
    __shared__ uint64_t bars[1 + 2 * ST + 5 * NT];
    __shared__ uint32_t tmem_base_slot;

    const int warp = ptx::uniform_warp_idx(), lane = threadIdx.x & 31;
    const int item = blockIdx.x / prm.H, head = blockIdx.x % prm.H;
    const int2 it = prm.items[item];
    const int ev0 = prm.offsets[it.x], ev1 = prm.offsets[it.x + 1];
    const int q0 = ev0 + (it.y & 0xffffff) * ATT_BQ;                 // item = (event, first query tile | tiles << 24)
    if (q0 >= ev1) return;      // the host sized the work list from the event's row count INCLUDING pad rows (an upper bound)
    const int nt = min(min(NT, it.y >> 24), (ev1 - q0 + ATT_BQ - 1) / ATT_BQ);   // query tiles of this CTA that hold rows of the event (>= 1)
    const int nkv = (ev1 - ev0 + ATT_BK - 1) / ATT_BK;              // 64-key tiles
    const int nst = (ev1 - ev0 + ATT_SK - 1) / ATT_SK;              // 128-key TMA stages
    const uint32_t* valid_bits = (prm.valid_bits && !(prm.n_valid && prm.n_valid[it.x] == ev1 - ev0)) ? prm.valid_bits : nullptr;

    const uint32_t smem_base = (ptx::smem_u32(smem_raw) + 1023u) & ~1023u;
    const uint32_t sQ = smem_base;                                  // Q tiles
    const uint32_t sKV = smem_base + NT * Cfg::Q_BYTES;
    const uint32_t sOnes = sKV + ST * Cfg::STAGE_BYTES;
    const uint32_t bar_q = ptx::smem_u32(&bars[0]);
    const uint32_t bar_kv_full = ptx::smem_u32(&bars[1]);
    const uint32_t bar_kv_empty = ptx::smem_u32(&bars[1 + ST]);
    const uint32_t bar_s = ptx::smem_u32(&bars[1 + 2 * ST]);             // [2t + b]: S_t(j) landed in buffer b = j & 1
    const uint32_t bar_p = ptx::smem_u32(&bars[1 + 2 * ST + 2 * NT]);    // [2t + b]: P_t(j) written over buffer b
    const uint32_t bar_o = ptx::smem_u32(&bars[1 + 2 * ST + 4 * NT]);    // [t]: O_t(j) complete

    if (warp == Cfg::WARP_TMA && lane == 0) {
        ptx::mbar_init(bar_q, 1);
        for (int s = 0; s < ST; ++s) {
            ptx::mbar_init(bar_kv_full + 8 * s, 1);
            ptx::mbar_init(bar_kv_empty + 8 * s, nt);                // one commit per active query tile
        }
        for (int i = 0; i < 2 * NT; ++i) {
            ptx::mbar_init(bar_s + 8 * i, 1);
            ptx::mbar_init(bar_p + 8 * i, 4);                        // one arrival per softmax warp
        }
        for (int i = 0; i < NT; ++i) ptx::mbar_init(bar_o + 8 * i, 1);
        ptx::fence_barrier_init();
        ptx::tma_prefetch_desc(&tmQKV);
    }
    if (warp == Cfg::WARP_MMA) {
        ptx::tmem_alloc(ptx::smem_u32(&tmem_base_slot), 512);
        ptx::tmem_relinquish();
    }
    if (warp < 4 * NT) {
        for (int i = threadIdx.x; i < Cfg::ONES_BYTES / 4; i += 4 * NT * 32)
            asm volatile("st.shared.b32 [%0], %1;" ::"r"(sOnes + 4 * i), "r"(0x3f803f80u) : "memory");
        ptx::fence_proxy_async();                                    // generic-proxy writes -> visible to the MMA
    }
    ptx::tc_fence_before();
    __syncthreads();
    ptx::tc_fence_after();
    const uint32_t tmem_base = tmem_base_slot;

    if (warp >= 4 * NT) {
    ptx::setmaxnreg_dec<Cfg::PRODUCER_REGS>();
    if (warp == Cfg::WARP_TMA) {
        // ------------------------------------------------------------ TMA producer
        if (lane == 0) {
            ptx::mbar_expect_tx(bar_q, Cfg::Q_BYTES * nt);
            for (int t = 0; t < nt; ++t) ptx::tma_load_2d(sQ + t * Cfg::Q_BYTES, &tmQKV, bar_q, head * HD, q0 + t * ATT_BQ);
        }
        for (int i = 0; i < nst; ++i) {
            const int s = i % ST;
            ptx::mbar_wait_long(bar_kv_empty + 8 * s, ((i / ST) & 1) ^ 1);
            if (lane == 0) {
                const uint32_t st = sKV + s * Cfg::STAGE_BYTES;
                const int k0 = ev0 + i * ATT_SK;
                ptx::mbar_expect_tx(bar_kv_full + 8 * s, Cfg::STAGE_BYTES);
                ptx::tma_load_2d(st, &tmQKV, bar_kv_full + 8 * s, prm.d + head * HD, k0);
                ptx::tma_load_2d(st + Cfg::K_BYTES, &tmQKV, bar_kv_full + 8 * s, 2 * prm.d + head * HD, k0);
            }
            __syncwarp();
        }
    } else if (warp - Cfg::WARP_MMA < nt) {
        // ------------------------------------------------------------ MMA issuers (one per query tile)
        const int t = warp - Cfg::WARP_MMA;
        constexpr uint32_t idesc_s = ptx::umma_idesc_bf16(128, ATT_BK);
        constexpr uint32_t idesc_o = ptx::umma_idesc_bf16(128, HD) | ptx::UMMA_B_MN_MAJOR;
        constexpr uint32_t idesc_l = ptx::umma_idesc_bf16(128, 8);
        constexpr uint32_t HALF = ATT_BK * Cfg::SW;                  // bytes of a 64-key half of a K or V stage
        auto issue_s = [&](int j) {                 // S_t(j) = Q_t K_j^T -> S buffer j & 1
            const uint32_t kb = sKV + ((j >> 1) % ST) * Cfg::STAGE_BYTES + (j & 1) * HALF;
            const uint32_t qb = sQ + t * Cfg::Q_BYTES;
#pragma unroll
            for (int k = 0; k < HD / 16; ++k)
                ptx::mma_ss(tmem_base + 128 * t + 64 * (j & 1), ptx::umma_desc_kmajor(qb + k * 32, Cfg::SW),
                            ptx::umma_desc_kmajor(kb + k * 32, Cfg::SW), idesc_s, k != 0);
            ptx::mma_commit(bar_s + 8 * (2 * t + (j & 1)));
        };
        auto issue_o = [&](int j) {                 // O_t += P_t(j) V_j (accumulated in TMEM over all key tiles)
            const uint32_t vb = sKV + ((j >> 1) % ST) * Cfg::STAGE_BYTES + Cfg::K_BYTES + (j & 1) * HALF;
#pragma unroll
            for (int k = 0; k < ATT_BK / 16; ++k)
                ptx::mma_ts(tmem_base + Cfg::O_COL0 + Cfg::OW * t, tmem_base + 128 * t + 64 * (j & 1) + k * 8,
                            ptx::umma_desc_mnmajor(vb + k * 16 * Cfg::SW, Cfg::SW), idesc_o, (j | k) != 0);
            const uint64_t ones = ptx::umma_desc_kmajor(sOnes, 128);      // row sums l_t += P_t(j) 1 next to O_t
#pragma unroll
            for (int k = 0; k < ATT_BK / 16; ++k)
                ptx::mma_ts(tmem_base + Cfg::O_COL0 + Cfg::OW * t + HD, tmem_base + 128 * t + 64 * (j & 1) + k * 8, ones, idesc_l,
                            (j | k) != 0);
            ptx::mma_commit(bar_o + 8 * t);
        };
        ptx::mbar_wait(bar_q, 0);
        ptx::mbar_wait(bar_kv_full, 0);
        ptx::tc_fence_after();
        issue_s(0);                                  // all lanes: one is elected inside the MMA / commit wrappers
        if (nkv > 1) issue_s(1);
        for (int j = 0; j < nkv; ++j) {
            ptx::mbar_wait_long(bar_p + 8 * (2 * t + (j & 1)), (j >> 1) & 1);     // P_t(j) is in TMEM
            ptx::tc_fence_after();
            issue_o(j);
            // K and V of stage j >> 1 are no longer needed by this tile after its second half
            if ((j & 1) || j == nkv - 1) ptx::mma_commit(bar_kv_empty + 8 * ((j >> 1) % ST));
            if (j + 2 < nkv) {                       // S_t(j+2) reuses S buffer j & 1: in order after P_t(j) V_j
                const int i2 = (j + 2) >> 1;
                if (((j + 2) & 1) == 0) ptx::mbar_wait(bar_kv_full + 8 * (i2 % ST), (i2 / ST) & 1);
                ptx::tc_fence_after();
                issue_s(j + 2);
            }
        }
    }
    } else {
        // ------------------------------------------------------------ softmax warpgroups
        ptx::setmaxnreg_inc<Cfg::SOFTMAX_REGS>();
        const int t = warp >> 2;                       // query tile of this warpgroup
        const int q = warp & 3;                        // TMEM lane quarter this warp may access
        const int qrow = q0 + t * ATT_BQ + q * 32 + lane;
        if (t < nt) {
            const uint32_t lane_addr = tmem_base + ((uint32_t)(q * 32) << 16);
            const uint32_t o_addr = lane_addr + Cfg::O_COL0 + Cfg::OW * t;
            const float c = prm.scale_log2;
            float m_ref = -INFINITY;
            // O_t *= corr in TMEM (all 32 lanes of the warp, rows that did not move have corr = 1): only when the
            // warp's reference maximum moved, which happens a few times per row (lazy rescaling)
            auto rescale_o = [&](float corr) {
                const float2 c2 = make_float2(corr, corr);
                uint32_t lsum;
                ptx::tmem_ld1(o_addr + HD, lsum);                 // the row sum (column hd; columns hd+1.. are copies)
#pragma unroll
                for (int c0 = 0; c0 < HD; c0 += 32) {
                    constexpr int CH = HD < 32 ? HD : 32;
                    uint32_t r[CH];
#pragma unroll
                    for (int w = 0; w < CH / 16; ++w) ptx::tmem_ld16(o_addr + c0 + w * 16, *reinterpret_cast<uint32_t(*)[16]>(&r[w * 16]));
                    ptx::tmem_ld_wait();
#pragma unroll
                    for (int i = 0; i < CH / 2; ++i) {
                        const float2 v = ptx::fmul2(make_float2(__uint_as_float(r[2 * i]), __uint_as_float(r[2 * i + 1])), c2);
                        r[2 * i] = __float_as_uint(v.x); r[2 * i + 1] = __float_as_uint(v.y);
                    }
#pragma unroll
                    for (int w = 0; w < CH / 16; ++w) ptx::tmem_st16(o_addr + c0 + w * 16, *reinterpret_cast<uint32_t(*)[16]>(&r[w * 16]));
                    if (c0 == 0) ptx::tmem_st1(o_addr + HD, __float_as_uint(__uint_as_float(lsum) * corr));
                }
            };
            // scores of the current tile live in registers; the next tile's are loaded while this one is finished
            uint32_t s[64];
            auto load_s = [&](int j) {
                ptx::mbar_wait(bar_s + 8 * (2 * t + (j & 1)), (j >> 1) & 1);
                ptx::tc_fence_after();
                const uint32_t s_addr = lane_addr + 128 * t + 64 * (j & 1);
                ptx::tmem_ld32(s_addr, *reinterpret_cast<uint32_t(*)[32]>(&s[0]));
                ptx::tmem_ld32(s_addr + 32, *reinterpret_cast<uint32_t(*)[32]>(&s[32]));
            };
            load_s(0);
            ptx::tmem_ld_wait();
            // one key tile; MASKED is a compile-time tag so that the loop over full tiles of pad-free events contains no
            // masking code at all (with both variants inside one loop body the unmasked path ran 9 % slower: measured)
            auto tile = [&](int j, auto masked_tag) {
                constexpr bool MASKED = decltype(masked_tag)::value;
                uint32_t mask[2] = {0xffffffffu, 0xffffffffu};
                if (MASKED) {   // 64 bits = (key inside the event) & (valid row), from the schedule's bit array
                    const int k0 = ev0 + j * ATT_BK;
                    const int left = min(ev1 - k0, ATT_BK);                     // 1 .. 64 keys of the event in this tile
                    mask[0] = left >= 32 ? 0xffffffffu : (1u << left) - 1u;
                    mask[1] = left >= 64 ? 0xffffffffu : (left <= 32 ? 0u : (1u << (left - 32)) - 1u);
                    if (valid_bits) {
                        const uint32_t* wp = valid_bits + (k0 >> 5);            // warp-uniform loads
                        const uint32_t w0 = __ldg(wp), w1 = __ldg(wp + 1), w2 = __ldg(wp + 2);
                        mask[0] &= __funnelshift_r(w0, w1, k0 & 31);
                        mask[1] &= __funnelshift_r(w1, w2, k0 & 31);
                    }
                }
                const uint32_t s_addr = lane_addr + 128 * t + 64 * (j & 1);
                bool rescale;
                float corr;
                if (MASKED && HD == 64) corr = softmax_tile_mask_once(s, s_addr, mask, c, m_ref, rescale);
                else corr = softmax_tile<!MASKED>(s, s_addr, mask, c, m_ref, rescale);
                // S_t(j+1) was issued after P_t(j-1) V_(j-1) and the tensor pipe completes in order: once S_t(j+1) has
                // landed, O_t holds all products up to j-1.  Only the last tile has to wait on bar_o for that.
                if (j + 1 < nkv) {
                    ptx::mbar_wait(bar_s + 8 * (2 * t + ((j + 1) & 1)), ((j + 1) >> 1) & 1);   // usually long complete
                } else if (j > 0) {
                    ptx::mbar_wait(bar_o + 8 * t, (j - 1) & 1);
                }
                ptx::tc_fence_after();
                if (rescale && j > 0) rescale_o(corr);    // before P_t(j) is published: no MMA is writing O_t now
                if (j + 1 < nkv) {                        // next tile's scores: in flight while the P stores drain
                    const uint32_t s_next = lane_addr + 128 * t + 64 * ((j + 1) & 1);
                    ptx::tmem_ld32(s_next, *reinterpret_cast<uint32_t(*)[32]>(&s[0]));
                    ptx::tmem_ld32(s_next + 32, *reinterpret_cast<uint32_t(*)[32]>(&s[32]));
                }
                ptx::tmem_st_wait();
                ptx::tc_fence_before();
                __syncwarp();
                if (lane == 0) ptx::mbar_arrive(bar_p + 8 * (2 * t + (j & 1)));      // P_t(j) (and the rescaled O_t) are in TMEM
                ptx::tmem_ld_wait();
            };
            int j = 0;
            if (!valid_bits) {                            // pad-free event: every tile but a ragged last one is full
                const int n_full = (ev1 - ev0) / ATT_BK;
                for (; j < n_full; ++j) tile(j, std::false_type{});
            }
            for (; j < nkv; ++j) tile(j, std::true_type{});
            // all products are in: O_t -> registers, normalise, store
            ptx::mbar_wait(bar_o + 8 * t, (nkv - 1) & 1);
            ptx::tc_fence_after();
            uint32_t o_r[HD];
#pragma unroll
            for (int w = 0; w < HD / 16; ++w) ptx::tmem_ld16(o_addr + w * 16, *reinterpret_cast<uint32_t(*)[16]>(&o_r[w * 16]));
            uint32_t lsum;
            ptx::tmem_ld1(o_addr + HD, lsum);
            ptx::tmem_ld_wait();
            if (qrow < ev1) {
                const float l_run = __uint_as_float(lsum);
                const float inv = l_run > 0.0f ? 1.0f / l_run : 0.0f;
                uint32_t hi[HD / 2], lo[HD / 2];
#pragma unroll
                for (int i = 0; i < HD / 2; ++i) {
                    const float y0 = __uint_as_float(o_r[2 * i]) * inv, y1 = __uint_as_float(o_r[2 * i + 1]) * inv;
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
    if (warp == Cfg::WARP_MMA) ptx::tmem_dealloc(tmem_base, 512);
}

template <int HD>
static int tc_attn_launch_hd(TcContext* c, const bf16* QKV, int64_t N, AttnParams prm, cudaStream_t st) {
    using Cfg = AttnCfg<HD>;
    CUtensorMap tmQKV;
    if (tc_tensor_map(c, &tmQKV, QKV, 3 * prm.d, N, 3 * prm.d, HD, ATT_SK)) return -1;
    auto kern = k_tc_attn<HD>;
    if (tc_set_smem_attr(c, (const void*)kern, Cfg::SMEM_BYTES)) return -1;
    kern<<<prm.n_items * prm.H, Cfg::THREADS, Cfg::SMEM_BYTES, st>>>(tmQKV, prm);
    return 0;
}

// items: (event, group index) pairs, one per CTA-row-group of tc_attn_rows_per_cta(hd) query rows
int tc_attn_launch(TcContext* c, const bf16* QKV, int64_t N, const uint32_t* valid_bits, const int* n_valid,
                          const int* offsets, const int2* items, int n_items, int d, int H, bf16* O, bf16* O_lo,
                          cudaStream_t st) {
    const int hd = d / H;
    AttnParams prm;
    prm.valid_bits = valid_bits; prm.n_valid = n_valid; prm.offsets = offsets; prm.items = items; prm.n_items = n_items;
    prm.H = H; prm.d = d; prm.O = O; prm.O_lo = O_lo;
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
