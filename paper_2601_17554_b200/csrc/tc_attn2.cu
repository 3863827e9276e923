// tc_attn2.cu -- varlen, key-padding-masked flash-attention forward on tcgen05 / TMEM / TMA (sm_100a), second design.
// Step a4 of DESIGN.md:  per event, per head  O = softmax(Q K^T / sqrt(hd) + mask) V   (Eq. 4), without
// the n x n matrix ever leaving the SM (L154).  Keys outside the event or of pad rows get weight exactly 0 (reading A2);
// a query with no valid key gets O = 0 (A15).
//
// What differs from tc_attn.cu (round 1): the softmax needs NO running maximum.
//   Eq. 4 is invariant under subtracting any per-row constant from the scores.  Round 1 tracked the row maximum tile by
//   tile (one FMNMX per score, a warp vote per tile, an in-place rescale of O when it moved).  Here the constant is the
//   Cauchy-Schwarz bound  B_i = |q_i| max_j |k_j| / sqrt(hd)  >= max_j s_ij  taken from the row norms (a0-style
//   pre-pass k_attn_norms: |q_i| per row and head, max |k_j| per event and head).  P = 2^((s - B) c) <= 1 can never
//   overflow, bf16 P keeps its relative precision at any magnitude (8 exponent bits), and the row sums and O accumulate in
//   fp32, so the result does not depend on how loose the bound is -- as long as nothing underflows.  The largest term of
//   a row is at least 2^(-2 B c): with 2 B c <= 96 there are more than 24 bits of headroom above the flush-to-zero
//   threshold 2^-126 and the FAST path is exact to fp32 rounding.  A CTA whose rows have a larger bound (huge query/key
//   norms: never seen with LayerNorm-ed inputs, but inputs are not ours to choose) takes the EXACT path instead: one extra
//   sweep over the keys computes the true row maxima (scores only, no P, no P V), then the same loop runs with them.
// With no cross-score dependency left, a query row is split over TWO threads (two warps per TMEM lane quarter, 32 of a
// tile's 64 scores each): twice the warps for the same registers, which is what hides the TMEM-load / MUFU latency that
// bound round 1's kernel (0.32 of the bf16 peak with neither the MUFU nor the issue slots saturated).
//
// One CTA = one head x NT consecutive 128-row query tiles of one event (NT = 3 at hd <= 32, 2 at hd = 64) sharing every
// K / V tile.  Key tiles are 64 keys wide, S is double-buffered in TMEM:
//   warps 0 .. 8NT-1   softmax: warp w serves query tile t = w / 8, lane quarter q = w % 4, score half hf = (w / 4) % 2:
//               S[32 of 64 columns] -> P = 2^(s c - B c) as bf16 written back over the first 16 of ITS OWN 32 columns.
//   warp 8NT    TMA producer: Q tiles once; then stages of (K, V), [128 keys x hd] each, row-major boxes of the one
//               [N, 3d] QKV buffer (an event may start at any row).
//   warps 8NT+1 .. 8NT+NT   MMA issuers, one per query tile: S_t(j) = Q_t K_j^T (M 128, N 64, K hd);
//               O_t += P_t(j) V_j (A = P from TMEM, B = V_j MN-major) and l_t += P_t(j) 1 (row sums on the tensor pipe).
// TMEM columns: S_t[b] at 128 t + 64 b; O_t | l_t at 128 NT + (hd + 8) t.
#include "tc_api.h"
#include "ptx.cuh"
#include <type_traits>

namespace mlpf {

constexpr int A2_BQ = 128, A2_BK = 64, A2_SK = 128;     // query tile, key tile, keys per TMA stage
constexpr float A2_FAST_MAX_BOUND = 48.0f;              // fast path iff B c <= 48 (log2 units) for every row of the CTA

template <int HD>
struct Attn2Cfg {
    static constexpr int NT = HD <= 32 ? 3 : 2;
    static constexpr int SM_WARPS = 8 * NT;
    static constexpr int THREADS = SM_WARPS * 32 + 128;
    static constexpr int WARP_TMA = SM_WARPS, WARP_MMA = SM_WARPS + 1;
    static constexpr int Q_BYTES = A2_BQ * HD * 2;
    static constexpr int K_BYTES = A2_SK * HD * 2;
    static constexpr int STAGE_BYTES = 2 * K_BYTES;
    static constexpr int STAGES = HD == 64 ? 4 : 6;
    static constexpr int ONES_BYTES = 1024;
    static constexpr int OW = HD + 8;
    static constexpr int XCHG_BYTES = NT * A2_BQ * 2 * 4;   // exact path: the two score halves' row maxima
    static constexpr int SMEM_BYTES = NT * Q_BYTES + STAGES * STAGE_BYTES + ONES_BYTES + XCHG_BYTES + 1024;
    static constexpr int SW = HD * 2;
    static constexpr int O_COL0 = 128 * NT;
    static_assert(O_COL0 + NT * OW <= 512, "TMEM budget");
};

int tc_attn2_rows_per_cta(int hd) { return (hd <= 32 ? 3 : 2) * A2_BQ; }

struct Attn2Params {
    const uint32_t* valid_bits; const int* n_valid; const int* offsets; const int2* items;
    const float* qn;           // [N, H] |q_i| per head
    const float* kmax;         // [E, H] max_j |k_j| over the event's rows, per head
    int n_items, H, d;
    bf16* O; bf16* O_lo;
    float scale_log2;          // c = log2(e) / sqrt(hd)
    int force_exact;           // debugging / tests: every CTA takes the exact path
};

// ---------------------------------------------------------------------------------------------- norms pre-pass
// qn[i, h] = |q_i| (head h), kmax[e, h] = max over the rows of event e of |k_j| (float bits, atomicMax on ints: norms
// are non-negative).  One thread per (row, head); a block's threads that belong to the block's first event reduce in
// shared memory first.  kmax must be zeroed before the launch.
__global__ void __launch_bounds__(256)
k_attn_norms(const bf16* __restrict__ QKV, const int* __restrict__ row_event, int N, int H, int hd, int d,
             const int* __restrict__ nc_dev, int group_rows, float* __restrict__ qn, float* __restrict__ kmax) {
    __shared__ int smax[64];
    __shared__ int ev_first;
    const int idx = blockIdx.x * blockDim.x + threadIdx.x;
    const int row = idx / H, h = idx % H;
    if (threadIdx.x < 64) smax[threadIdx.x] = 0;
    if (threadIdx.x == 0) ev_first = row_event[min(row, N - 1)];
    __syncthreads();
    // pad-row compaction: rows at or beyond the number of meaningful rows (of their stack) hold stale data and stale event
    // ids: they must not leak into kmax (the bound, and with it the rounding of P, would depend on the buffer's history)
    const int nc = nc_dev ? __ldg(nc_dev) : 0x7fffffff;
    if (row < N && (group_rows > 0 ? row % group_rows : row) < nc) {
        const uint4* qp = reinterpret_cast<const uint4*>(QKV + (int64_t)row * 3 * d + h * hd);
        const uint4* kp = reinterpret_cast<const uint4*>(QKV + (int64_t)row * 3 * d + d + h * hd);
        float sq = 0.f, sk = 0.f;
        for (int i = 0; i < hd / 8; ++i) {
            const uint4 a = __ldg(qp + i), b = __ldg(kp + i);
            const uint32_t aw[4] = {a.x, a.y, a.z, a.w}, bw[4] = {b.x, b.y, b.z, b.w};
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                const float a0 = __uint_as_float(aw[k] << 16), a1 = __uint_as_float(aw[k] & 0xffff0000u);
                const float b0 = __uint_as_float(bw[k] << 16), b1 = __uint_as_float(bw[k] & 0xffff0000u);
                sq = fmaf(a0, a0, fmaf(a1, a1, sq));
                sk = fmaf(b0, b0, fmaf(b1, b1, sk));
            }
        }
        qn[(int64_t)row * H + h] = sqrtf(sq);
        const int kb = __float_as_int(sqrtf(sk));
        const int ev = row_event[row];
        if (ev == ev_first && h < 64) atomicMax(&smax[h], kb);
        else atomicMax(reinterpret_cast<int*>(kmax) + (int64_t)ev * H + h, kb);
    }
    __syncthreads();
    if ((int)threadIdx.x < H && threadIdx.x < 64 && smax[threadIdx.x] > 0)
        atomicMax(reinterpret_cast<int*>(kmax) + (int64_t)ev_first * H + threadIdx.x, smax[threadIdx.x]);
}

// 2^(s c - Bc) for a pair of scores on the FMA / ALU pipes instead of the MUFU (Cody-Waite split + degree-3 polynomial, max
// relative error 1.0e-4, 40x below the bf16 rounding of P).  Bc is an INTEGER (the bound rounded up), so everything the
// range reduction needs comes out of exactly rounded FMAs on the raw scores:
//   xr = s c + (M - Bc)            M = 1.5 * 2^23: the low mantissa bits of xr hold n = round(s c - Bc)
//   f  = s c - (Bc + n)            with Bc + n = xr - (M - Bc) exactly;  |f| <= 0.5
//   2^f ~ 1 + f (c1 + f (c2 + f c3));  2^n goes into the exponent field with one integer multiply-add.
// 8 issue slots per pair.  Fast path only (s c - Bc > -97 there); the exact path and masked tiles (-inf scores) use the MUFU.
__device__ __forceinline__ float2 a2_exp2_poly2(float2 sc, float2 c2, float2 k1) {
    const float2 xr = ptx::ffma2(sc, c2, k1);
    const float2 m = ptx::fadd2(xr, make_float2(-k1.x, -k1.y));
    const float2 f = ptx::ffma2(sc, c2, make_float2(-m.x, -m.y));
    float2 p = ptx::ffma2(f, make_float2(0.0550089306f, 0.0550089306f), make_float2(0.2422109596f, 0.2422109596f));
    p = ptx::ffma2(p, f, make_float2(0.6932829272f, 0.6932829272f));
    p = ptx::ffma2(p, f, make_float2(1.0f, 1.0f));
    return make_float2(__int_as_float(__float_as_int(p.x) + (__float_as_int(xr.x) << 23)),
                       __int_as_float(__float_as_int(p.y) + (__float_as_int(xr.y) << 23)));
}
// The same for scores that already carry the scale (PS, see the kernel) and need no offset: 2^s.
//   xr = s + M;  n = xr - M;  f = s - n  (all exact)
// (Tried: 2^n as a float from ONE funnel shift per value (M = 1.5 * 2^23 + 127, rotate xr left by 23 = K 2^n with the
// constant K = 1.2939453125 folded into the coefficients) and a final packed multiply, which moves the two integer
// multiply-adds from the FMA pipe to the idle ALU pipe: slower, 2.93 vs 2.87 ms per cfg3 step of attention.  The loop is
// bound by issue slots, two per packed or 16-lane instruction, not by any one pipe.)
// DEG = 2 (experiment, MLPF_OPT_ATTN_POLY_DEG): the minimax quadratic, max relative error 1.83e-3 = the size of P's own bf16
// rounding (2^-9), one packed FMA less per pair.
template <int DEG>
__device__ __forceinline__ float2 a2_exp2_poly2_ps(float2 s) {
    const float2 xr = ptx::fadd2(s, make_float2(12582912.0f, 12582912.0f));
    const float2 m = ptx::fadd2(xr, make_float2(-12582912.0f, -12582912.0f));
    const float2 f = ptx::fadd2(s, make_float2(-m.x, -m.y));
    float2 p;
    if (DEG == 2) {
        p = ptx::ffma2(f, make_float2(0.23864397f, 0.23864397f), make_float2(0.70388058f, 0.70388058f));
        p = ptx::ffma2(p, f, make_float2(1.00046145f, 1.00046145f));
    } else {
        p = ptx::ffma2(f, make_float2(0.0550089306f, 0.0550089306f), make_float2(0.2422109596f, 0.2422109596f));
        p = ptx::ffma2(p, f, make_float2(0.6932829272f, 0.6932829272f));
        p = ptx::ffma2(p, f, make_float2(1.0f, 1.0f));
    }
    return make_float2(__int_as_float(__float_as_int(p.x) + (__float_as_int(xr.x) << 23)),
                       __int_as_float(__float_as_int(p.y) + (__float_as_int(xr.y) << 23)));
}
// PE of every 16 pairs of exponentials run on the FMA pipe, evenly spread (PE = 0: all on the MUFU).  The MUFU does 16 ex2
// per clock and SM and is the binding unit at hd = 32 (one ex2 per 128 tensor FLOPs); PE balances the MUFU against the
// FMA / ALU pipes and the issue slots (measured on cfg3, ms per step of the attention class: profiles/r02_README.md).

// 32 scores of one row -> 16 packed bf16 pairs  p = 2^(s c - Bc).  MASKED: scores of masked keys become -inf first, so the
// MUFU gives the exact weight 0 (the polynomial path is not used on masked tiles).
// PS (pre-scaled scores, fast path): S already holds s c and no offset is subtracted (see the kernel): unmasked tiles feed
// the MUFU straight from TMEM; masked tiles and the exact path keep the FMA with c = 1.
template <bool MASKED, int PE, bool PS, int DEG = 3>
__device__ __forceinline__ void a2_exp32(uint32_t (&s)[32], uint32_t mask, float c, float neg_bc, uint32_t (&pk)[16]) {
    const float2 c2 = make_float2(c, c), m2 = make_float2(neg_bc, neg_bc);
    const float2 k1 = make_float2(12582912.0f + neg_bc, 12582912.0f + neg_bc);      // exact: neg_bc is an integer on this path
#pragma unroll
    for (int i = 0; i < 16; ++i) {
        if (MASKED) {
            s[2 * i] = (mask >> (2 * i)) & 1u ? s[2 * i] : 0xff800000u;
            s[2 * i + 1] = (mask >> (2 * i + 1)) & 1u ? s[2 * i + 1] : 0xff800000u;
        }
        const float2 sc = make_float2(__uint_as_float(s[2 * i]), __uint_as_float(s[2 * i + 1]));
        float2 p;
        if (!MASKED && ((i + 1) * PE) / 16 > (i * PE) / 16) p = PS ? a2_exp2_poly2_ps<DEG>(sc) : a2_exp2_poly2(sc, c2, k1);
        else if (!MASKED && PS) p = make_float2(ptx::fast_exp2(sc.x), ptx::fast_exp2(sc.y));
        else {
            const float2 x = ptx::ffma2(sc, c2, m2);
            p = make_float2(ptx::fast_exp2(x.x), ptx::fast_exp2(x.y));
        }
        __nv_bfloat162 b2 = __floats2bfloat162_rn(p.x, p.y);
        pk[i] = *reinterpret_cast<uint32_t*>(&b2);
    }
}

template <int HD, int PE, bool PS, int DEG = 3>
__global__ void __launch_bounds__(Attn2Cfg<HD>::THREADS, 1)
k_tc_attn2(const __grid_constant__ CUtensorMap tmQKV, Attn2Params prm) {
    using Cfg = Attn2Cfg<HD>;
    constexpr int ST = Cfg::STAGES, NT = Cfg::NT;
    extern __shared__ uint8_t smem_raw[];
    __shared__ uint64_t bars[2 + 2 * ST + 5 * NT];
    __shared__ uint32_t tmem_base_slot;
    __shared__ int bound_bits;                                   // max over the CTA's rows of B c (float bits)

    // programmatic dependent launch: this grid's first wave may be resident before the QKV projection has finished (the
    // work list decides whether a CTA exists at all, so the wait comes first)
    ptx::grid_dep_wait();
    ptx::grid_dep_launch();
    const int warp = ptx::uniform_warp_idx(), lane = threadIdx.x & 31;
    const int item = blockIdx.x / prm.H, head = blockIdx.x % prm.H;
    const int2 it = prm.items[item];
    const int ev0 = prm.offsets[it.x], ev1 = prm.offsets[it.x + 1];
    const int q0 = ev0 + (it.y & 0xffffff) * A2_BQ;               // item = (event, first query tile | tiles << 24)
    if (q0 >= ev1) return;      // the host sized the work list from the event's row count INCLUDING pad rows (an upper bound)
    const int nt = min(min(NT, it.y >> 24), (ev1 - q0 + A2_BQ - 1) / A2_BQ);
    const int nkv = (ev1 - ev0 + A2_BK - 1) / A2_BK;
    const int nst = (ev1 - ev0 + A2_SK - 1) / A2_SK;
    const uint32_t* valid_bits = (prm.valid_bits && !(prm.n_valid && prm.n_valid[it.x] == ev1 - ev0)) ? prm.valid_bits : nullptr;

    const uint32_t smem_base = (ptx::smem_u32(smem_raw) + 1023u) & ~1023u;
    const uint32_t sQ = smem_base;
    const uint32_t sKV = smem_base + NT * Cfg::Q_BYTES;
    const uint32_t sOnes = sKV + ST * Cfg::STAGE_BYTES;
    float* const xchg = reinterpret_cast<float*>(smem_raw + (smem_base - ptx::smem_u32(smem_raw)) + NT * Cfg::Q_BYTES +
                                                 ST * Cfg::STAGE_BYTES + Cfg::ONES_BYTES);
    const uint32_t bar_q = ptx::smem_u32(&bars[0]);
    const uint32_t bar_kv_full = ptx::smem_u32(&bars[1]);
    const uint32_t bar_kv_empty = ptx::smem_u32(&bars[1 + ST]);
    const uint32_t bar_s = ptx::smem_u32(&bars[1 + 2 * ST]);             // [2t + b]: S_t landed in buffer b
    const uint32_t bar_p = ptx::smem_u32(&bars[1 + 2 * ST + 2 * NT]);    // [2t + b]: P_t written over buffer b (or S consumed)
    const uint32_t bar_o = ptx::smem_u32(&bars[1 + 2 * ST + 4 * NT]);    // [t]: all of O_t accumulated
    const uint32_t bar_vc = ptx::smem_u32(&bars[1 + 2 * ST + 5 * NT]);   // the last V stage's foreign rows are zeroed
    // The last 128-row K / V stage of an event runs into the NEXT event's first rows.  Their keys get weight exactly 0 (masked
    // tile), but 0 x NaN = NaN in the P V product: a non-finite row of the next event would poison this event's accumulators.
    // The producer warp therefore zeroes those V rows in shared memory before the issuers may read the stage (once per CTA).
    const int last_rows = (ev1 - ev0) - (nst - 1) * A2_SK;                 // keys of this event in its last stage: 1 .. 128
    const bool v_clean = last_rows < A2_SK;

    if (threadIdx.x == 0) bound_bits = 0;
    if (warp == Cfg::WARP_TMA && lane == 0) {
        ptx::mbar_init(bar_q, 1);
        for (int s = 0; s < ST; ++s) {
            ptx::mbar_init(bar_kv_full + 8 * s, 1);
            ptx::mbar_init(bar_kv_empty + 8 * s, nt);
        }
        for (int i = 0; i < 2 * NT; ++i) {
            ptx::mbar_init(bar_s + 8 * i, 1);
            ptx::mbar_init(bar_p + 8 * i, 8);                        // one arrival per softmax warp of the tile
        }
        for (int i = 0; i < NT; ++i) ptx::mbar_init(bar_o + 8 * i, 1);
        ptx::mbar_init(bar_vc, 1);
        ptx::fence_barrier_init();
        // Q and the first ring of K / V stages go out at once: they do not depend on the fast / exact decision below, whose
        // global loads (row norms) would otherwise sit in front of the first TMA in every CTA's prologue
        ptx::mbar_expect_tx(bar_q, Cfg::Q_BYTES * nt);
        for (int t = 0; t < nt; ++t) ptx::tma_load_2d(sQ + t * Cfg::Q_BYTES, &tmQKV, bar_q, head * HD, q0 + t * A2_BQ);
        for (int g = 0; g < min(ST, nst); ++g) {
            const uint32_t st = sKV + g * Cfg::STAGE_BYTES;
            ptx::mbar_expect_tx(bar_kv_full + 8 * g, Cfg::STAGE_BYTES);
            ptx::tma_load_2d(st, &tmQKV, bar_kv_full + 8 * g, prm.d + head * HD, ev0 + g * A2_SK);
            ptx::tma_load_2d(st + Cfg::K_BYTES, &tmQKV, bar_kv_full + 8 * g, 2 * prm.d + head * HD, ev0 + g * A2_SK);
        }
    }
    if (warp == Cfg::WARP_MMA) {
        ptx::tmem_alloc(ptx::smem_u32(&tmem_base_slot), 512);
        ptx::tmem_relinquish();
    }
    __syncthreads();
    // softmax threads: the row's bound B c = |q_i| max|k| c, and its maximum over the CTA (decides fast / exact)
    const int t_sm = warp >> 3, q_sm = warp & 3, hf = (warp >> 2) & 1;
    const int qrow = q0 + t_sm * A2_BQ + q_sm * 32 + lane;
    float bc = 0.0f;
    if (warp < Cfg::SM_WARPS) {
        for (int i = threadIdx.x; i < Cfg::ONES_BYTES / 4; i += Cfg::SM_WARPS * 32)
            asm volatile("st.shared.b32 [%0], %1;" ::"r"(sOnes + 4 * i), "r"(0x3f803f80u) : "memory");
        ptx::fence_proxy_async();
        if (t_sm < nt && qrow < ev1) {
            bc = __ldg(prm.qn + (int64_t)qrow * prm.H + head) * __ldg(prm.kmax + (int64_t)it.x * prm.H + head) * (PS ? 1.0f : prm.scale_log2) * 1.008f;   // 2^-7: norms may come from the values before their bf16 rounding
            bc = ceilf(bc);                                          // an integer bound: the polynomial path's range reduction is exact
            if (!(bc >= 0.0f) || bc > 3.0e38f) bc = 3.0e38f;         // NaN / inf norms: exact path (which is NaN-transparent too)
        }
        const float wmax = warp_max(bc);
        if (lane == 0 && wmax > 0.0f) atomicMax(&bound_bits, __float_as_int(wmax));
    }
    ptx::tc_fence_before();
    __syncthreads();
    ptx::tc_fence_after();
    const uint32_t tmem_base = tmem_base_slot;
    const bool exact = prm.force_exact || __int_as_float(bound_bits) > A2_FAST_MAX_BOUND;
    const int n_sweeps = exact ? 2 : 1;          // exact: sweep 0 = row maxima only, sweep 1 = the softmax proper

    if (warp == Cfg::WARP_TMA) {
        // ------------------------------------------------------------ TMA producer
        for (int g = min(ST, nst); g < n_sweeps * nst; ++g) {        // g = running stage counter over both sweeps (the first ring is under way)
            const int s = g % ST, i = g % nst;
            ptx::mbar_wait_long(bar_kv_empty + 8 * s, ((g / ST) & 1) ^ 1);
            if (lane == 0) {
                const uint32_t st = sKV + s * Cfg::STAGE_BYTES;
                const int k0 = ev0 + i * A2_SK;
                ptx::mbar_expect_tx(bar_kv_full + 8 * s, Cfg::STAGE_BYTES);
                ptx::tma_load_2d(st, &tmQKV, bar_kv_full + 8 * s, prm.d + head * HD, k0);
                ptx::tma_load_2d(st + Cfg::K_BYTES, &tmQKV, bar_kv_full + 8 * s, 2 * prm.d + head * HD, k0);
            }
            __syncwarp();
        }
        if (v_clean) {                           // the softmax sweep's last stage has landed: zero V rows last_rows .. 127
            const int g = n_sweeps * nst - 1, s = g % ST;
            ptx::mbar_wait_long(bar_kv_full + 8 * s, (g / ST) & 1);
            const uint32_t vt = sKV + s * Cfg::STAGE_BYTES + Cfg::K_BYTES + last_rows * Cfg::SW;   // (a row's swizzled chunks stay inside the row)
            for (int i = lane; i < (A2_SK - last_rows) * Cfg::SW / 16; i += 32)
                asm volatile("st.shared.v4.b32 [%0], {%1, %1, %1, %1};" ::"r"(vt + 16 * i), "r"(0) : "memory");
            ptx::fence_proxy_async();
            __syncwarp();
            if (lane == 0) ptx::mbar_arrive(bar_vc);
        }
    } else if (warp > Cfg::WARP_TMA && warp - Cfg::WARP_MMA < nt) {
        // ------------------------------------------------------------ MMA issuers (one per query tile)
        const int t = warp - Cfg::WARP_MMA;
        constexpr uint32_t idesc_s = ptx::umma_idesc_bf16(128, A2_BK);
        constexpr uint32_t idesc_o = ptx::umma_idesc_bf16(128, HD) | ptx::UMMA_B_MN_MAJOR;
        constexpr uint32_t idesc_l = ptx::umma_idesc_bf16(128, 8);
        constexpr uint32_t HALF = A2_BK * Cfg::SW;
        // The issuer's own instructions compete with the softmax warps for the scheduler's issue slots (the kernel is issue
        // bound), so everything that depends on the running counters is kept incrementally: the stage of the current key
        // tile pair (index, parity, the low word of its K descriptor) and the S buffer; descriptors differ from one another
        // only by constants added to that low word (start address >> 4; no carry: shared memory is < 2^18 bytes).
        const uint32_t HI_K = (uint32_t)(ptx::umma_desc_kmajor(0, Cfg::SW) >> 32), LO_K = (uint32_t)ptx::umma_desc_kmajor(0, Cfg::SW);
        const uint32_t HI_V = (uint32_t)(ptx::umma_desc_mnmajor(0, Cfg::SW) >> 32), LO_V = (uint32_t)ptx::umma_desc_mnmajor(0, Cfg::SW);
        auto mk = [](uint32_t hi, uint32_t lo) { return ((uint64_t)hi << 32) | lo; };
        const uint32_t qd = (sQ + t * Cfg::Q_BYTES) >> 4;                       // Q_t, + 2 k per 16-column step
        const uint64_t ones = ptx::umma_desc_kmajor(sOnes, 128);
        const uint32_t s_t = tmem_base + 128 * t, o_t = tmem_base + Cfg::O_COL0 + Cfg::OW * t;
        const uint32_t bs_t = bar_s + 16 * t, bp_t = bar_p + 16 * t;
        // S_t(buffer b) = Q_t K^T for the key tile at shared-memory address (>> 4) kd
        auto issue_s = [&](uint32_t b, uint32_t kd) {
#pragma unroll
            for (int k = 0; k < HD / 16; ++k)
                ptx::mma_ss(s_t + 64 * b, mk(HI_K, LO_K | (qd + 2 * k)), mk(HI_K, LO_K | (kd + 2 * k)), idesc_s, k != 0);
            ptx::mma_commit(bs_t + 8 * b);
        };
        // O_t += P_t(buffer b) V, l_t += P_t(buffer b) 1 for the value tile at (>> 4) vd
        auto issue_o = [&](uint32_t b, uint32_t vd, bool first) {
#pragma unroll
            for (int k = 0; k < A2_BK / 16; ++k) {                  // keys 16k .. 16k+15: P columns 32 (k / 2) + 8 (k % 2)
                const uint32_t pa = s_t + 64 * b + 32 * (k >> 1) + 8 * (k & 1);
                ptx::mma_ts(o_t, pa, mk(HI_V, LO_V | (vd + k * Cfg::SW)), idesc_o, !(first && k == 0));
                ptx::mma_ts(o_t + HD, pa, ones, idesc_l, !(first && k == 0));
            }
        };
        constexpr uint32_t STG16 = Cfg::STAGE_BYTES >> 4, HALF16 = HALF >> 4, KB16 = Cfg::K_BYTES >> 4;
        ptx::mbar_wait(bar_q, 0);
        uint32_t stg = 0, stg_par = 0, kd = sKV >> 4;             // stage of the key tile pair that holds tile j
        uint32_t nb = 0, np = 0;                                  // S buffer n & 1 and parity (n >> 1) & 1 of tile j
        for (int sw = 0; sw < n_sweeps; ++sw) {
            const bool pv = sw == n_sweeps - 1;
            // the first two S tiles of the sweep (one stage)
            ptx::mbar_wait(bar_kv_full + 8 * stg, stg_par);
            ptx::tc_fence_after();
            issue_s(nb, kd);
            if (nkv > 1) issue_s(nb ^ 1u, kd + HALF16);
            for (int j = 0; j < nkv; ++j) {
                const uint32_t odd = (uint32_t)j & 1u;
                ptx::mbar_wait_long(bp_t + 8 * nb, np);                     // P_t(j) in TMEM (sweep 0 of 2: S consumed)
                ptx::tc_fence_after();
                if (pv && v_clean && (j >> 1) == nst - 1 && (!odd || j == 0)) {      // first tile of the last stage
                    ptx::mbar_wait_long(bar_vc, 0);
                    ptx::tc_fence_after();
                }
                if (pv) issue_o(nb, kd + KB16 + odd * HALF16, j == 0);
                const bool last_of_stage = odd || j == nkv - 1;
                if (last_of_stage) ptx::mma_commit(bar_kv_empty + 8 * stg);
                // the stage after this one
                uint32_t stg2 = stg + 1, par2 = stg_par, kd2 = kd + STG16;
                if (stg2 == (uint32_t)ST) { stg2 = 0; par2 ^= 1u; kd2 = sKV >> 4; }
                if (j + 2 < nkv) {                   // S_t(j+2) reuses this S buffer: in order after P_t(j) V_j
                    if (!odd) ptx::mbar_wait(bar_kv_full + 8 * stg2, par2);
                    ptx::tc_fence_after();
                    issue_s(nb, kd2 + odd * HALF16);
                }
                if (last_of_stage) { stg = stg2; stg_par = par2; kd = kd2; }
                np ^= nb; nb ^= 1u;                  // n + 1
            }
        }
        ptx::mma_commit(bar_o + 8 * t);
    } else if (warp < Cfg::SM_WARPS) {
        // ------------------------------------------------------------ softmax warps
        const int t = t_sm, q = q_sm;
        if (t < nt) {
            const uint32_t lane_addr = tmem_base + ((uint32_t)(q * 32) << 16);
            const uint32_t o_addr = lane_addr + Cfg::O_COL0 + Cfg::OW * t;
            // PS: q was multiplied by c = log2(e) / sqrt(hd) before its bf16 rounding (QKV projection's epilogue), so S = s c.
            // On the fast path |s c| <= B c <= 48 then bounds P = 2^(s c) to [2^-48, 2^48] by itself: nothing is subtracted at
            // all (bf16 P and the fp32 sums have the exponent range for it; O / l cancels any common factor).
            const float c = PS ? 1.0f : prm.scale_log2;
            // 32-bit mask of this warp's score half of key tile j: (key inside the event) & (valid row)
            auto tile_mask = [&](int j) -> uint32_t {
                const int k0 = ev0 + j * A2_BK + 32 * hf;
                const int left = ev1 - k0;                               // may be <= 0
                uint32_t m = left >= 32 ? 0xffffffffu : (left <= 0 ? 0u : (1u << left) - 1u);
                if (valid_bits) {
                    const uint32_t* wp = valid_bits + (k0 >> 5);
                    m &= __funnelshift_r(__ldg(wp), __ldg(wp + 1), k0 & 31);
                }
                return m;
            };
            // (the exact path sends EVERY tile through the masked variant: its exponents can be far below -126)
            const int n_full = valid_bits ? 0 : (ev1 - ev0 - 32 * hf + 32) / A2_BK;   // leading tiles whose half [64 j + 32 hf, + 32) lies inside the event
            int n = 0;
            float neg_bc = PS ? 0.0f : -bc;
            if (exact) {
                // sweep 0: the true row maximum over the valid keys (scores only)
                float mx = -INFINITY;
                for (int j = 0; j < nkv; ++j, ++n) {
                    ptx::mbar_wait(bar_s + 8 * (2 * t + (n & 1)), (n >> 1) & 1);
                    ptx::tc_fence_after();
                    uint32_t s[32];
                    ptx::tmem_ld32(lane_addr + 128 * t + 64 * (n & 1) + 32 * hf, s);
                    ptx::tmem_ld_wait();
                    const uint32_t m = tile_mask(j);
                    float m4[4] = {mx, -INFINITY, -INFINITY, -INFINITY};
#pragma unroll
                    for (int i = 0; i < 32; ++i) m4[i & 3] = fmaxf(m4[i & 3], (m >> i) & 1u ? __uint_as_float(s[i]) : -INFINITY);
                    mx = fmaxf(fmaxf(m4[0], m4[1]), fmaxf(m4[2], m4[3]));
                    ptx::tc_fence_before();
                    __syncwarp();
                    if (lane == 0) ptx::mbar_arrive(bar_p + 8 * (2 * t + (n & 1)));      // S consumed
                }
                // the row's two score halves exchange their maxima
                xchg[(t * A2_BQ + q * 32 + lane) * 2 + hf] = mx;
                asm volatile("bar.sync %0, 64;" ::"r"(1 + t * 4 + q) : "memory");
                mx = fmaxf(mx, xchg[(t * A2_BQ + q * 32 + lane) * 2 + (hf ^ 1)]);
                neg_bc = (mx == -INFINITY) ? 0.0f : -mx * c;
            }
            // the softmax sweep.  tile_at: one key tile with everything that depends on the S buffer passed in (barrier
            // addresses, TMEM address, parity), so that the main loop, unrolled over the two buffers, carries no per-tile
            // address arithmetic (the loop is issue-bound: 126 instructions per 32 scores before, ~100 of them arithmetic)
            auto tile_at = [&](uint32_t b_s, uint32_t b_p, uint32_t s_addr, uint32_t par, int j, auto masked_tag) {
                constexpr bool MASKED = decltype(masked_tag)::value;
                ptx::mbar_wait(b_s, par);
                ptx::tc_fence_after();
                uint32_t s[32], pk[16];
                ptx::tmem_ld32(s_addr, s);
                const uint32_t m = MASKED ? tile_mask(j) : 0xffffffffu;
                ptx::tmem_ld_wait();
                a2_exp32<MASKED, PE, PS, DEG>(s, m, c, neg_bc, pk);
                ptx::tmem_st16(s_addr, pk);
                ptx::tmem_st_wait();
                ptx::tc_fence_before();
                __syncwarp();
                if (lane == 0) ptx::mbar_arrive(b_p);
            };
            auto tile = [&](int j, auto masked_tag) {
                tile_at(bar_s + 8 * (2 * t + (n & 1)), bar_p + 8 * (2 * t + (n & 1)), lane_addr + 128 * t + 64 * (n & 1) + 32 * hf,
                        (n >> 1) & 1, j, masked_tag);
            };
            {
                int j = 0;
                const int jf = exact ? 0 : n_full;
                if ((n & 1) && j < jf) { tile(j, std::false_type{}); ++j; ++n; }
                const uint32_t bs0 = bar_s + 8 * (2 * t), bp0 = bar_p + 8 * (2 * t), sa0 = lane_addr + 128 * t + 32 * hf;
                uint32_t par = (n >> 1) & 1;
                for (; j + 1 < jf; j += 2, n += 2, par ^= 1u) {
                    tile_at(bs0, bp0, sa0, par, j, std::false_type{});
                    tile_at(bs0 + 8, bp0 + 8, sa0 + 64, par, j + 1, std::false_type{});
                }
                for (; j < jf; ++j, ++n) tile(j, std::false_type{});
                for (; j < nkv; ++j, ++n) tile(j, std::true_type{});
            }
            // all products are in: this warp's half of O_t -> registers, normalise, store
            ptx::mbar_wait(bar_o + 8 * t, 0);
            ptx::tc_fence_after();
            constexpr int HW = HD / 2;                                  // output columns of this warp
            uint32_t o_r[HW];
#pragma unroll
            for (int w = 0; w < HW / 8; ++w) {
                if (HW % 16 == 0 && (w & 1) == 0) ptx::tmem_ld16(o_addr + HW * hf + w * 8, *reinterpret_cast<uint32_t(*)[16]>(&o_r[w * 8]));
                if (HW % 16 != 0) {
#pragma unroll
                    for (int i = 0; i < 8; ++i) ptx::tmem_ld1(o_addr + HW * hf + w * 8 + i, o_r[w * 8 + i]);
                }
            }
            uint32_t lsum;
            ptx::tmem_ld1(o_addr + HD, lsum);
            ptx::tmem_ld_wait();
            if (qrow < ev1) {
                const float l_run = __uint_as_float(lsum);
                const float inv = l_run > 0.0f ? 1.0f / l_run : 0.0f;
                uint32_t hi[HW / 2], lo[HW / 2];
#pragma unroll
                for (int i = 0; i < HW / 2; ++i) {
                    const float y0 = __uint_as_float(o_r[2 * i]) * inv, y1 = __uint_as_float(o_r[2 * i + 1]) * inv;
                    __nv_bfloat162 h2 = __floats2bfloat162_rn(y0, y1);
                    hi[i] = *reinterpret_cast<uint32_t*>(&h2);
                    __nv_bfloat162 l2 = __floats2bfloat162_rn(y0 - __low2float(h2), y1 - __high2float(h2));
                    lo[i] = *reinterpret_cast<uint32_t*>(&l2);
                }
                uint4* op = reinterpret_cast<uint4*>(prm.O + (int64_t)qrow * prm.d + head * HD + HW * hf);
#pragma unroll
                for (int i = 0; i < HW / 8; ++i) op[i] = make_uint4(hi[4 * i], hi[4 * i + 1], hi[4 * i + 2], hi[4 * i + 3]);
                if (prm.O_lo) {
                    uint4* lp = reinterpret_cast<uint4*>(prm.O_lo + (int64_t)qrow * prm.d + head * HD + HW * hf);
#pragma unroll
                    for (int i = 0; i < HW / 8; ++i) lp[i] = make_uint4(lo[4 * i], lo[4 * i + 1], lo[4 * i + 2], lo[4 * i + 3]);
                }
            }
        }
    }
    ptx::tc_fence_before();
    __syncthreads();
    if (warp == Cfg::WARP_MMA) ptx::tmem_dealloc(tmem_base, 512);
}

int g_attn2_poly_deg = 3;            // tuning knob (MLPF_OPT_ATTN_POLY_DEG): 3 (default) | 2
int g_attn2_poly_every = -1;          // tuning knob (MLPF_OPT_ATTN_POLY): -1 = the default of the head dimension

template <int HD, int PE, bool PS, int DEG = 3>
static int tc_attn2_launch_pe(TcContext* c, const bf16* QKV, int64_t N, Attn2Params prm, cudaStream_t st) {
    using Cfg = Attn2Cfg<HD>;
    CUtensorMap tmQKV;
    if (tc_tensor_map(c, &tmQKV, QKV, 3 * prm.d, N, 3 * prm.d, HD, A2_SK)) return -1;
    auto kern = k_tc_attn2<HD, PE, PS, DEG>;
    if (tc_set_smem_attr(c, (const void*)kern, Cfg::SMEM_BYTES)) return -1;
    tc_launch(kern, dim3(prm.n_items * prm.H), dim3(Cfg::THREADS), Cfg::SMEM_BYTES, st, c->pdl, tmQKV, prm);
    return 0;
}

template <int HD, bool PS>
static int tc_attn2_launch_hd(TcContext* c, const bf16* QKV, int64_t N, Attn2Params prm, cudaStream_t st) {
    // measured (profiles/r02_README.md): with prescaled scores 8 of 16 at every head dimension (hd = 64: 4.41 -> 3.37 ms of
    // attention per cfg5a step against all-MUFU); the unscaled form (kernel-level entry) keeps its own optimum
    const int pe = g_attn2_poly_every >= 0 ? g_attn2_poly_every : (PS ? 8 : (HD == 64 ? 0 : 7));
    if (PS && g_attn2_poly_deg == 2) {            // experiment: quadratic polynomial (prescaled scores only)
        switch (pe) {
            case 9: return tc_attn2_launch_pe<HD, 9, PS, 2>(c, QKV, N, prm, st);
            default: return tc_attn2_launch_pe<HD, 8, PS, 2>(c, QKV, N, prm, st);
        }
    }
    switch (pe) {
        case 0: return tc_attn2_launch_pe<HD, 0, PS>(c, QKV, N, prm, st);
        case 4: return tc_attn2_launch_pe<HD, 4, PS>(c, QKV, N, prm, st);
        case 8: return tc_attn2_launch_pe<HD, 8, PS>(c, QKV, N, prm, st);
        case 9: return tc_attn2_launch_pe<HD, 9, PS>(c, QKV, N, prm, st);
        default: return tc_attn2_launch_pe<HD, 7, PS>(c, QKV, N, prm, st);
    }
}

// norms pre-pass + attention.  qn [N, H] and kmax [E, H] are caller-owned scratch; row_event [N] from the schedule.
int tc_attn2_launch(TcContext* c, const bf16* QKV, int64_t N, int E, const uint32_t* valid_bits, const int* n_valid,
                    const int* offsets, const int* row_event, const int2* items, int n_items, int d, int H, float* qn,
                    float* kmax, bf16* O, bf16* O_lo, int force_exact, const int* nc_dev, int group_rows, cudaStream_t st,
                    bool norms_ready, bool prescaled) {
    const int hd = d / H;
    if (H > 64) { snprintf(c->err, sizeof c->err, "tc_attn2: more than 64 heads"); return -1; }
    if (!norms_ready) {                      // (the model path gets qn / kmax from the QKV projection's epilogue instead)
        cudaMemsetAsync(kmax, 0, (size_t)E * H * 4, st);
        const int64_t nthr = N * H;
        k_attn_norms<<<(unsigned)((nthr + 255) / 256), 256, 0, st>>>(QKV, row_event, (int)N, H, hd, d, nc_dev, group_rows, qn, kmax);
    }
    Attn2Params prm;
    prm.valid_bits = valid_bits; prm.n_valid = n_valid; prm.offsets = offsets; prm.items = items; prm.n_items = n_items;
    prm.qn = qn; prm.kmax = kmax; prm.H = H; prm.d = d; prm.O = O; prm.O_lo = O_lo; prm.force_exact = force_exact;
    prm.scale_log2 = 1.4426950408889634f / sqrtf((float)hd);
    switch (hd) {     // prescaled: the q columns of QKV already carry the factor log2(e) / sqrt(hd) (and qn is the norm of those)
        case 16: return prescaled ? tc_attn2_launch_hd<16, true>(c, QKV, N, prm, st) : tc_attn2_launch_hd<16, false>(c, QKV, N, prm, st);
        case 32: return prescaled ? tc_attn2_launch_hd<32, true>(c, QKV, N, prm, st) : tc_attn2_launch_hd<32, false>(c, QKV, N, prm, st);
        case 64: return prescaled ? tc_attn2_launch_hd<64, true>(c, QKV, N, prm, st) : tc_attn2_launch_hd<64, false>(c, QKV, N, prm, st);
    }
    snprintf(c->err, sizeof c->err, "tc_attn2: head_dim %d unsupported", hd);
    return -1;
}

}  // namespace mlpf
