// tc_heads.cu -- step a8 as ONE tcgen05 / TMEM / TMA kernel (sm_100a): all two-layer FFN heads ("six two-layer
// FFN heads"; readings A11 / A12) of a 128-row tile, hidden layers kept on chip:
//   hid_b = act(z W1[b]^T + b1[b])   for head block b (hidden width d);   out[:, outputs of b] = hid_b W2[b]^T + b2[b]
// i.e. an FFN whose second layer is block-diagonal.  Same machinery as tc_post.cu: z (bf16 hi + lo) is a resident shared-
// memory A operand; per 128-column chunk of the stacked hidden layer  S_b = z W1[chunk]^T  lands in one of two TMEM
// buffers, the epilogue warps add b1, apply the activation and write the hidden values BACK over S as packed bf16
// (hi | lo per 32-column group); the second MMA takes them as its A operand straight from TMEM against a 16-row tile of
// W2 (the block's output rows as bf16 hi + lo, zero-padded to 16), accumulating into 16 TMEM columns per head block.
// The hidden layer (5 d values per element, hi + lo) never reaches HBM; round 1 wrote and re-read it (252 MB on cfg3).
// Rows are compacted rows; the final epilogue scatters to the original rows (orig_row), pad rows were zeroed beforehand.
// D = d_model in {64, 128, 256}.  Warps: 0 = TMA producer, 1 = MMA issuer, 2..17 = epilogue (thread = row).
#include "tc_api.h"
#include "ptx.cuh"
#include "epi_math.cuh"

namespace mlpf {

constexpr int HD_BM = 128, HD_SLOT = 16384, HD_THREADS = 576, HD_NS = 5;

template <int D>
struct HeadsCfg {
    static constexpr int KB = D / 64;
    static constexpr int CH = D < 128 ? D : 128;          // hidden columns per chunk
    static constexpr int CPB = D / CH;                    // chunks per head block
    static constexpr int NCG = CH / 32;                   // 32-column groups per chunk = epilogue warps per lane quarter at work
    static constexpr int A_BYTES = 2 * KB * HD_SLOT;
    static int smem_bytes(int nblk) { return A_BYTES + HD_NS * HD_SLOT + nblk * D * 4 + 1024; }
};

struct HeadsParams {
    int M, nblk, chunk0;            // rows; head blocks of this launch; first chunk (row offset into W1 / W2p in chunks)
    const int* nc_dev;
    const float* b1;                // [nblk * D] first-layer biases of this launch's blocks
    const float* b2;                // [n_out] output biases (all outputs)
    const int* orig_row;            // compacted row -> original row (null: identity)
    int out_of[16 * MAX_HBLK];      // accumulator column 16 * (block - first block) + j -> global output index, -1: unused
    HeadsOut ho;
    float *out_logits, *out_regress, *out_binary;
};

template <int D, int ACT>
__global__ void __launch_bounds__(HD_THREADS, 1)
k_tc_heads(const __grid_constant__ CUtensorMap tmZ, const __grid_constant__ CUtensorMap tmZlo,
           const __grid_constant__ CUtensorMap tmW1, const __grid_constant__ CUtensorMap tmW2, HeadsParams p) {
    using Cfg = HeadsCfg<D>;
    constexpr int KB = Cfg::KB, CH = Cfg::CH, CPB = Cfg::CPB, NCG = Cfg::NCG, NS = HD_NS;
    extern __shared__ uint8_t smem_raw[];
    __shared__ uint64_t bars[2 * NS + 8];
    __shared__ uint32_t tmem_base_slot;

    const int warp = ptx::uniform_warp_idx(), lane = threadIdx.x & 31;
    const int n_tiles = (p.M + HD_BM - 1) / HD_BM;
    const int NC = p.nblk * CPB;
    int nc_rows = 0x7fffffff;                  // (read after the set-up, behind grid_dep_wait)
    auto skip_tile = [&](int tile) { return tile * HD_BM >= nc_rows; };
    const uint32_t smem_base = (ptx::smem_u32(smem_raw) + 1023u) & ~1023u;
    uint8_t* const smem_gen = smem_raw + (smem_base - ptx::smem_u32(smem_raw));
    const uint32_t sA = smem_base, sRing = sA + Cfg::A_BYTES;
    float* const v_b1 = reinterpret_cast<float*>(smem_gen + Cfg::A_BYTES + NS * HD_SLOT);
    const uint32_t bar_full = ptx::smem_u32(&bars[0]), bar_empty = ptx::smem_u32(&bars[NS]);
    const uint32_t bar_a_full = ptx::smem_u32(&bars[2 * NS]), bar_a_free = bar_a_full + 8, bar_s_full = bar_a_full + 16 /* [2] */,
                   bar_g = bar_a_full + 32 /* [2] */, bar_acc_final = bar_a_full + 48, bar_acc_free = bar_a_full + 56;

    if (warp == 0 && lane == 0) {
        for (int s = 0; s < NS; ++s) { ptx::mbar_init(bar_full + 8 * s, 1); ptx::mbar_init(bar_empty + 8 * s, 1); }
        ptx::mbar_init(bar_a_full, 1); ptx::mbar_init(bar_a_free, 1);
        for (int b = 0; b < 2; ++b) { ptx::mbar_init(bar_s_full + 8 * b, 1); ptx::mbar_init(bar_g + 8 * b, 4 * NCG); }
        ptx::mbar_init(bar_acc_final, 1); ptx::mbar_init(bar_acc_free, 4);
        ptx::fence_barrier_init();
        ptx::tma_prefetch_desc(&tmZ); ptx::tma_prefetch_desc(&tmZlo); ptx::tma_prefetch_desc(&tmW1); ptx::tma_prefetch_desc(&tmW2);
    }
    if (warp == 1) {
        ptx::tmem_alloc(ptx::smem_u32(&tmem_base_slot), 512);
        ptx::tmem_relinquish();
    }
    for (int i = threadIdx.x; i < p.nblk * D; i += HD_THREADS) v_b1[i] = __ldg(p.b1 + i);     // (weights: not the predecessor's)
    ptx::tc_fence_before();
    __syncthreads();
    ptx::tc_fence_after();
    const uint32_t tmem_base = tmem_base_slot;
    // programmatic dependent launch: the set-up above may overlap the previous kernel's tail; nothing below may
    ptx::grid_dep_wait();
    ptx::grid_dep_launch();
    if (p.nc_dev) nc_rows = __ldg(p.nc_dev);

    if (warp == 0) {
        // ------------------------------------------------------------ TMA producer
        uint32_t slot_it = 0;
        auto acquire = [&]() -> uint32_t {
            const uint32_t s = slot_it % NS;
            ptx::mbar_wait(bar_empty + 8 * s, ((slot_it / NS) & 1) ^ 1);
            ++slot_it;
            return s;
        };
        auto load_w1 = [&](int c) {                         // KB slots of [CH rows x 64 k]
            for (int kb = 0; kb < KB; ++kb) {
                const uint32_t s = acquire();
                if (lane == 0) {
                    ptx::mbar_expect_tx(bar_full + 8 * s, CH * 128);
                    ptx::tma_load_2d(sRing + s * HD_SLOT, &tmW1, bar_full + 8 * s, kb * 64, (p.chunk0 + c) * CH);
                }
                __syncwarp();
            }
        };
        auto load_w2 = [&](int c) {                         // one slot: [hi | lo] x (CH / 64 k-blocks) boxes of [16 rows x 64 k]
            const uint32_t s = acquire();
            if (lane == 0) {
                ptx::mbar_expect_tx(bar_full + 8 * s, 2 * (CH / 64) * 2048);
                for (int hl = 0; hl < 2; ++hl)
                    for (int kb = 0; kb < CH / 64; ++kb)
                        ptx::tma_load_2d(sRing + s * HD_SLOT + (hl * (CH / 64) + kb) * 2048, &tmW2, bar_full + 8 * s, kb * 64,
                                         ((p.chunk0 + c) * 2 + hl) * 16);
            }
            __syncwarp();
        };
        int it = -1;
        for (int tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
            if (skip_tile(tile)) continue;
            ++it;
            const int m0 = tile * HD_BM;
            if (it > 0) ptx::mbar_wait(bar_a_free, (it - 1) & 1);
            if (lane == 0) {
                ptx::mbar_expect_tx(bar_a_full, Cfg::A_BYTES);
                for (int kb = 0; kb < KB; ++kb) {
                    ptx::tma_load_2d(sA + kb * HD_SLOT, &tmZ, bar_a_full, kb * 64, m0);
                    ptx::tma_load_2d(sA + (KB + kb) * HD_SLOT, &tmZlo, bar_a_full, kb * 64, m0);
                }
            }
            __syncwarp();
            load_w1(0);
            if (NC > 1) load_w1(1);
            for (int c = 0; c < NC; ++c) {
                load_w2(c);
                if (c + 2 < NC) load_w1(c + 2);
            }
        }
    } else if (warp == 1) {
        // ------------------------------------------------------------ MMA issuer
        constexpr uint32_t idesc_s = ptx::umma_idesc_bf16(HD_BM, CH);
        constexpr uint32_t idesc_o = ptx::umma_idesc_bf16(HD_BM, 16);
        uint32_t slot_it = 0, ph_g = 0;
        auto wait_slot = [&]() -> uint32_t {
            const uint32_t s = slot_it % NS;
            ptx::mbar_wait(bar_full + 8 * s, (slot_it / NS) & 1);
            ptx::tc_fence_after();
            return sRing + s * HD_SLOT;
        };
        auto free_slot = [&]() { ptx::mma_commit(bar_empty + 8 * (slot_it % NS)); ++slot_it; };
        int it = -1;
        for (int tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
            if (skip_tile(tile)) continue;
            ++it;
            ptx::mbar_wait(bar_a_full, it & 1);
            if (it > 0) ptx::mbar_wait(bar_acc_free, (it - 1) & 1);
            ptx::tc_fence_after();
            auto mma1 = [&](int c) {                         // S_(c&1) = z W1[chunk c]^T (hi + lo)
                const uint32_t sb = tmem_base + 256 + 128 * (c & 1);
                for (int kb = 0; kb < KB; ++kb) {
                    const uint32_t b = wait_slot();
#pragma unroll
                    for (int k = 0; k < 4; ++k) {
                        const uint64_t bd = ptx::umma_desc_kmajor(b + k * 32, 128);
                        ptx::mma_ss(sb, ptx::umma_desc_kmajor(sA + kb * HD_SLOT + k * 32, 128), bd, idesc_s, (kb | k) != 0);
                        ptx::mma_ss(sb, ptx::umma_desc_kmajor(sA + (KB + kb) * HD_SLOT + k * 32, 128), bd, idesc_s, 1);
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
                ptx::mbar_wait(bar_g + 8 * bsel, (ph_g >> bsel) & 1);
                ph_g ^= 1u << bsel;
                ptx::tc_fence_after();
                const uint32_t gb = tmem_base + 256 + 128 * bsel;
                const uint32_t acc = tmem_base + 16 * (c / CPB);         // this head block's 16 output columns
                const uint32_t b = wait_slot();
#pragma unroll
                for (int j = 0; j < CH / 16; ++j) {                      // 16-wide k-steps of the chunk
                    const uint32_t off = (j >> 2) * 2048 + (j & 3) * 32;
                    const uint64_t bhi = ptx::umma_desc_kmajor(b + off, 128), blo = ptx::umma_desc_kmajor(b + (CH / 64) * 2048 + off, 128);
                    const uint32_t a_hi = gb + 32 * (j >> 1) + 8 * (j & 1);
                    ptx::mma_ts(acc, a_hi, bhi, idesc_o, ((c % CPB) | j) != 0);
                    ptx::mma_ts(acc, a_hi + 16, bhi, idesc_o, 1);
                    ptx::mma_ts(acc, a_hi, blo, idesc_o, 1);
                }
                free_slot();
                if (c + 2 < NC) {
                    mma1(c + 2);
                    if (c + 3 == NC) ptx::mma_commit(bar_a_free);
                }
            }
            ptx::mma_commit(bar_acc_final);
        }
    } else {
        // ------------------------------------------------------------ epilogue warps
        const int ew = warp - 2, q = warp & 3, cg = ew >> 2;
        const int r = q * 32 + lane;
        const uint32_t lane_addr = tmem_base + ((uint32_t)(q * 32) << 16);
        uint32_t ph_s = 0;
        int it = -1;
        for (int tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
            if (skip_tile(tile)) continue;
            ++it;
            const int row = tile * HD_BM + r;
            const bool row_ok = row < p.M && row < nc_rows;
            if (cg < NCG) {
                for (int c = 0; c < NC; ++c) {
                    const int bsel = c & 1;
                    ptx::mbar_wait(bar_s_full + 8 * bsel, (ph_s >> bsel) & 1);
                    ph_s ^= 1u << bsel;
                    ptx::tc_fence_after();
                    const uint32_t s_addr = lane_addr + 256 + 128 * bsel + 32 * cg;
                    uint32_t sv[32];
                    ptx::tmem_ld32(s_addr, sv);
                    ptx::tmem_ld_wait();
                    const float* bp = v_b1 + c * CH + 32 * cg;
                    uint32_t hi[16], lo[16];
#pragma unroll
                    for (int i = 0; i < 8; ++i) {
                        const float4 bb = *reinterpret_cast<const float4*>(bp + 4 * i);
                        float2 x0 = ptx::fadd2(make_float2(__uint_as_float(sv[4 * i]), __uint_as_float(sv[4 * i + 1])), make_float2(bb.x, bb.y));
                        float2 x1 = ptx::fadd2(make_float2(__uint_as_float(sv[4 * i + 2]), __uint_as_float(sv[4 * i + 3])), make_float2(bb.z, bb.w));
                        split_bf16x2(act2<ACT>(x0), hi[2 * i], lo[2 * i]);
                        split_bf16x2(act2<ACT>(x1), hi[2 * i + 1], lo[2 * i + 1]);
                    }
                    ptx::tmem_st16(s_addr, hi);
                    ptx::tmem_st16(s_addr + 16, lo);
                    ptx::tmem_st_wait();
                    ptx::tc_fence_before();
                    __syncwarp();
                    if (lane == 0) ptx::mbar_arrive(bar_g + 8 * bsel);
                }
            }
            if (cg == 0) {          // one warp per lane quarter: the tile's outputs -> original rows
                ptx::mbar_wait(bar_acc_final, it & 1);
                ptx::tc_fence_after();
                const int orow = (row_ok && p.orig_row) ? __ldg(p.orig_row + row) : row;
#pragma unroll
                for (int b = 0; b < MAX_HBLK; ++b) {                     // one head block (16 accumulator columns) at a time
                    if (b < p.nblk) {
                        uint32_t a[16];
                        ptx::tmem_ld16(lane_addr + 16 * b, a);
                        ptx::tmem_ld_wait();
                        if (row_ok) {
#pragma unroll
                            for (int j = 0; j < 16; ++j) {
                                const int o = p.out_of[16 * b + j];      // uniform (kernel parameter)
                                if (o >= 0) {
                                    const float v = __uint_as_float(a[j]) + __ldg(p.b2 + o);
                                    if (o < p.ho.n_bin) { if (p.out_binary) p.out_binary[orow] = v; }
                                    else if (o < p.ho.n_bin + p.ho.n_cls) p.out_logits[(int64_t)orow * p.ho.n_cls + (o - p.ho.n_bin)] = v;
                                    else p.out_regress[(int64_t)orow * p.ho.n_reg + (o - p.ho.n_bin - p.ho.n_cls)] = v;
                                }
                            }
                        }
                    }
                }
                ptx::tc_fence_before();
                __syncwarp();
                if (lane == 0) ptx::mbar_arrive(bar_acc_free);
            }
        }
    }
    ptx::tc_fence_before();
    __syncthreads();
    if (warp == 1) ptx::tmem_dealloc(tmem_base, 512);
}

// ------------------------------------------------------------------------------------------------ launch
bool tc_heads_supported(int d, int n_hblk) {
    if (d != 64 && d != 128 && d != 256) return false;
    if (n_hblk < 1 || n_hblk > MAX_HBLK) return false;
    const int smem = d == 64 ? HeadsCfg<64>::smem_bytes(n_hblk) : d == 128 ? HeadsCfg<128>::smem_bytes(n_hblk) : HeadsCfg<256>::smem_bytes(n_hblk);
    return smem + 512 <= 232448;
}
int tc_heads_chunk(int d) { return d < 128 ? d : 128; }

template <int D, int ACT>
static int tc_heads_launch_t(TcContext* c, const HeadsArgs& a, cudaStream_t st) {
    using Cfg = HeadsCfg<D>;
    CUtensorMap tmZ, tmZlo, tmW1, tmW2;
    if (tc_tensor_map(c, &tmZ, a.z, D, a.M, D, 64, HD_BM)) return -1;
    if (tc_tensor_map(c, &tmZlo, a.z_lo, D, a.M, D, 64, HD_BM)) return -1;
    if (tc_tensor_map(c, &tmW1, a.W1, D, (uint64_t)a.n_hblk_total * D, D, 64, Cfg::CH)) return -1;
    if (tc_tensor_map(c, &tmW2, a.W2p, Cfg::CH, (uint64_t)a.n_hblk_total * Cfg::CPB * 32, Cfg::CH, 64, 16)) return -1;
    auto kern = k_tc_heads<D, ACT>;
    if (tc_set_smem_attr(c, (const void*)kern, 232448 - 1024)) return -1;
    HeadsParams p;
    p.M = a.M; p.nblk = a.nblk; p.chunk0 = a.blk0 * Cfg::CPB; p.nc_dev = a.nc_dev;
    p.b1 = a.b1 + (int64_t)a.blk0 * D; p.b2 = a.b2; p.orig_row = a.orig_row; p.ho = a.ho;
    p.out_logits = a.out_logits; p.out_regress = a.out_regress; p.out_binary = a.out_binary;
    for (int k = 0; k < 16 * MAX_HBLK; ++k) p.out_of[k] = -1;
    int idx[MAX_HBLK] = {0};
    for (int o = 0; o < a.ho.n_out; ++o) {
        const int b = a.ho.blk[o];
        if (b >= a.blk0 && b < a.blk0 + a.nblk) p.out_of[16 * (b - a.blk0) + idx[b - a.blk0]++] = o;
    }
    const int n_tiles = (a.M + HD_BM - 1) / HD_BM;
    const int grid = n_tiles < c->num_sms ? n_tiles : c->num_sms;
    tc_launch(kern, dim3(grid), dim3(HD_THREADS), Cfg::smem_bytes(a.nblk), st, c->pdl, tmZ, tmZlo, tmW1, tmW2, p);
    return 0;
}

int tc_heads_launch(TcContext* c, const HeadsArgs& a, cudaStream_t st) {
    if (!tc_heads_supported(a.d, a.n_hblk_total) || a.nblk < 1 || a.blk0 + a.nblk > a.n_hblk_total || !a.z || !a.z_lo ||
        (a.act != ACT_GELU && a.act != ACT_RELU)) {
        snprintf(c->err, sizeof c->err, "tc_heads: unsupported shape d=%d blocks=%d act=%d", a.d, a.n_hblk_total, a.act);
        return -1;
    }
#define HEADS_CASE(DD) \
    if (a.d == DD) return a.act == ACT_GELU ? tc_heads_launch_t<DD, ACT_GELU>(c, a, st) : tc_heads_launch_t<DD, ACT_RELU>(c, a, st);
    HEADS_CASE(64) HEADS_CASE(128) HEADS_CASE(256)
#undef HEADS_CASE
    return -1;
}

}  // namespace mlpf
