// simple_kernels.cu -- CUDA-core kernels of libmlpf.so.
//  * the integer schedule (step a0), the embedding's first layer (a1), LayerNorm (a2) and the heads'
//    output layer (a8) are used by every path;
//  * the tiled FFMA GEMM and the one-thread-per-query attention are the fp32 debug path
//    (MLPF_PREC_FP32_DEBUG, parity <= 1e-4) and the MLPF_KERNELS_SIMPLE debugging aid in bf16.
// Citations are /root/reference/PAPER.md lines; readings A* are listed in DESIGN.md.
#include "simple_api.h"
#include <vector>
#include <cuda_fp8.h>

namespace mlpf {

// ------------------------------------------------------------------------------------------------
// a0: integer schedule on the device (the type id lives in device memory: reading A1)
// ------------------------------------------------------------------------------------------------

__device__ __forceinline__ int element_type(const float* __restrict__ X, int64_t row, int F) {
    float x0 = X[row * F];
    int t = (x0 >= 0.0f && x0 < 5.0f) ? (int)x0 : (x0 >= 5.0f ? 4 : 0);   // clamp to 0..4; NaN -> 0
    return t;
}

// per 1024-row block: histogram of types 0..4; also valid[], row_event[], row_pos[], n_valid[e] (atomic)
__global__ void __launch_bounds__(SCHED_BLOCK)
k_sched_count(const float* __restrict__ X, int N, int F, const int* __restrict__ offsets, int E,
              int* __restrict__ block_counts, int* __restrict__ valid, uint32_t* __restrict__ valid_bits,
              int* __restrict__ row_event, int* __restrict__ row_pos, int* __restrict__ n_valid) {
    __shared__ int hist[5];
    if (threadIdx.x < 5) hist[threadIdx.x] = 0;
    __syncthreads();
    int i = blockIdx.x * SCHED_BLOCK + threadIdx.x;
    int t = -1, ev = -1;
    if (i < N) {
        t = element_type(X, i, F);
        valid[i] = (t != 0);
        // event of row i: largest e with offsets[e] <= i  (offsets non-decreasing; empty events skipped)
        int lo = 0, hi = E;             // invariant: offsets[lo] <= i < offsets[hi]
        while (hi - lo > 1) {
            int mid = (lo + hi) >> 1;
            if (offsets[mid] <= i) lo = mid; else hi = mid;
        }
        row_event[i] = lo;
        row_pos[i] = i - offsets[lo];
        ev = lo;
    }
    {   // one bit per row, 32 rows per word (rows >= N: 0): the attention kernel's key mask
        const unsigned vb = __ballot_sync(0xffffffffu, t > 0);
        if ((threadIdx.x & 31) == 0) valid_bits[i >> 5] = vb;
        // n_valid: one atomic per (warp, event) instead of one per row (49 k same-address atomics took 30 us on cfg3)
        const unsigned grp = __match_any_sync(0xffffffffu, ev);
        const int cnt = __popc(grp & vb);
        if (ev >= 0 && cnt && (int)(threadIdx.x & 31) == __ffs(grp) - 1) atomicAdd(&n_valid[ev], cnt);
    }
#pragma unroll
    for (int ty = 0; ty < 5; ++ty) {
        unsigned m = __ballot_sync(0xffffffffu, t == ty);
        if ((threadIdx.x & 31) == 0 && m) atomicAdd(&hist[ty], __popc(m));
    }
    __syncthreads();
    if (threadIdx.x < 5) block_counts[blockIdx.x * 5 + threadIdx.x] = hist[threadIdx.x];
}

// one block: exclusive scan of the per-block counts per type; segment starts padded to 128 rows.  Thread 5: the same
// scan over the valid rows of all types (pad-row compaction): block_vbase[b] = valid rows before block b, n_comp[0] = total
__global__ void k_sched_scan(const int* __restrict__ block_counts, int nb, int* __restrict__ block_base,
                             int* __restrict__ type_offsets, int* __restrict__ block_vbase, int* __restrict__ n_comp) {
    __shared__ int total[5];
    int ty = threadIdx.x;
    if (ty < 5) {
        int run = 0;
        for (int b = 0; b < nb; ++b) {
            block_base[b * 5 + ty] = run;
            run += block_counts[b * 5 + ty];
        }
        total[ty] = run;
    } else if (ty == 5) {
        int run = 0;
        for (int b = 0; b < nb; ++b) {
            block_vbase[b] = run;
            run += block_counts[b * 5 + 1] + block_counts[b * 5 + 2] + block_counts[b * 5 + 3] + block_counts[b * 5 + 4];
        }
        n_comp[0] = run;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        int pos = 0;
        type_offsets[0] = 0;
        for (int t = 1; t <= 4; ++t) {
            type_offsets[t] = pos;
            pos += (total[t] + 127) / 128 * 128;
        }
        type_offsets[5] = pos;
    }
}

// stable counting sort by type: sorted_row[i] = slot, type_perm[slot] = i  (type_perm pre-filled with -1)
// Pad-row compaction (same pass): vbefore[i] = valid rows before row i; comp_row[i] = that
// number for a valid row, -1 for a pad row; orig_row / row_event_c = the inverse map and the event of a compacted row;
// comp_type_perm[slot] = compacted row of the slot's row.
__global__ void __launch_bounds__(SCHED_BLOCK)
k_sched_scatter(const float* __restrict__ X, int N, int F, const int* __restrict__ block_base,
                const int* __restrict__ type_offsets, const int* __restrict__ block_vbase, const int* __restrict__ row_event,
                int* __restrict__ sorted_row, int* __restrict__ type_perm, int* __restrict__ vbefore, int* __restrict__ comp_row,
                int* __restrict__ orig_row, int* __restrict__ row_event_c, int* __restrict__ comp_type_perm) {
    __shared__ int warp_cnt[32][5];
    int i = blockIdx.x * SCHED_BLOCK + threadIdx.x;
    int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    int t = (i < N) ? element_type(X, i, F) : -1;
    int my_rank = 0;
#pragma unroll
    for (int ty = 0; ty < 5; ++ty) {
        unsigned m = __ballot_sync(0xffffffffu, t == ty);
        if (t == ty) my_rank = __popc(m & ((1u << lane) - 1u));
        if (lane == 0) warp_cnt[w][ty] = __popc(m);
    }
    const unsigned mv = __ballot_sync(0xffffffffu, t > 0);
    const int vrank = __popc(mv & ((1u << lane) - 1u));
    __syncthreads();
    if (i < N) {
        int before_v = 0;
        for (int ww = 0; ww < w; ++ww) before_v += warp_cnt[ww][1] + warp_cnt[ww][2] + warp_cnt[ww][3] + warp_cnt[ww][4];
        const int comp = block_vbase[blockIdx.x] + before_v + vrank;
        vbefore[i] = comp;
        comp_row[i] = t > 0 ? comp : -1;
        if (t == 0) {
            sorted_row[i] = -1;
        } else {
            orig_row[comp] = i;
            row_event_c[comp] = row_event[i];
            int before = 0;
            for (int ww = 0; ww < w; ++ww) before += warp_cnt[ww][t];
            int slot = type_offsets[t] + block_base[blockIdx.x * 5 + t] + before + my_rank;
            sorted_row[i] = slot;
            type_perm[slot] = i;
            comp_type_perm[slot] = comp;
        }
    }
}

// offsets_c[e] = valid rows before the first row of event e (e = 0 .. E; offsets[E] = N)
__global__ void k_sched_offsets_c(const int* __restrict__ offsets, int E, int N, const int* __restrict__ vbefore,
                                  const int* __restrict__ n_comp, int* __restrict__ offsets_c) {
    for (int e = blockIdx.x * blockDim.x + threadIdx.x; e <= E; e += gridDim.x * blockDim.x) {
        const int o = offsets[e];
        offsets_c[e] = o < N ? vbefore[o] : n_comp[0];
    }
}

// ------------------------------------------------------------------------------------------------
// a1 (first layer): h1[slot] = act(W1[t] x + b1[t]) in fp32 on CUDA cores (raw features span
// 1e-2..1e4), rows written in by-type sorted order so that the second layer is a grouped GEMM.
// Pad rows (type 0): the residual stream row h[i,:] is set to exactly 0 (reading A2).
// W1t is [T][64][d] (k-major, zero padded to 64 features) so loads are coalesced over the d outputs.
// ------------------------------------------------------------------------------------------------

// 128 threads, each owning TWO output columns (j and j + d/2) with both weight columns in registers: every broadcast
// LDS.128 of a row's features feeds 8 FMAs instead of 4 (the one-column form was bound by shared-memory operand
// bandwidth: a 128-bit broadcast load costs 4 LSU cycles), two rows per pass for independent FMA chains.
constexpr int EMB_THREADS = 128;
template <typename T>
__global__ void __launch_bounds__(EMB_THREADS, 3)
k_embed_l1(const float* __restrict__ X, int N, int F, int d, const float* __restrict__ W1t,
           const float* __restrict__ b1, int act, const int* __restrict__ sorted_row,
           T* __restrict__ h1, T* __restrict__ h1_lo, float* __restrict__ h) {
    __shared__ __align__(16) float xs[EMB_ROWS][64];        // rows are read as broadcast 128-bit loads (no padding needed)
    __shared__ int list[5][EMB_ROWS];
    __shared__ int cnt[5];
    const int row0 = blockIdx.x * EMB_ROWS;
    const int rows = min(EMB_ROWS, N - row0);
    if (threadIdx.x < 5) cnt[threadIdx.x] = 0;
    for (int idx = threadIdx.x; idx < EMB_ROWS * 64; idx += EMB_THREADS) {
        int r = idx >> 6, k = idx & 63;
        xs[r][k] = (r < rows && k < F) ? X[(int64_t)(row0 + r) * F + k] : 0.0f;
    }
    __syncthreads();
    if (threadIdx.x < rows) {
        int t = element_type(X, row0 + threadIdx.x, F);
        int p = atomicAdd(&cnt[t], 1);
        list[t][p] = threadIdx.x;
    }
    __syncthreads();
    // pad rows -> zero residual-stream rows
    for (int p = 0; h && p < cnt[0]; ++p) {                  // (h == nullptr: compacted rows, pad rows do not exist there)
        int r = list[0][p];
        for (int j = threadIdx.x; j < d; j += EMB_THREADS) h[(int64_t)(row0 + r) * d + j] = 0.0f;
    }
    const int dh = d >> 1;
    for (int t = 1; t <= 4; ++t) {
        const int c = cnt[t];
        if (c == 0) continue;
        for (int j = threadIdx.x; j < dh; j += EMB_THREADS) {
            float wa[64], wb[64];
            const float* wp = W1t + ((int64_t)(t - 1) * 64) * d + j;
#pragma unroll
            for (int k = 0; k < 64; ++k) { wa[k] = wp[(int64_t)k * d]; wb[k] = wp[(int64_t)k * d + dh]; }
            const float bja = b1[(t - 1) * d + j], bjb = b1[(t - 1) * d + j + dh];
            for (int p = 0; p < c; p += 2) {
                const int r0 = list[t][p], r1 = list[t][min(p + 1, c - 1)];
                float a0 = bja, a1 = bja, c0 = bjb, c1 = bjb;
                const float4* x0 = reinterpret_cast<const float4*>(xs[r0]);
                const float4* x1 = reinterpret_cast<const float4*>(xs[r1]);
#pragma unroll
                for (int k = 0; k < 16; ++k) {
                    const float4 u = x0[k], v = x1[k];
                    a0 = fmaf(wa[4 * k], u.x, a0); a0 = fmaf(wa[4 * k + 1], u.y, a0);
                    a0 = fmaf(wa[4 * k + 2], u.z, a0); a0 = fmaf(wa[4 * k + 3], u.w, a0);
                    c0 = fmaf(wb[4 * k], u.x, c0); c0 = fmaf(wb[4 * k + 1], u.y, c0);
                    c0 = fmaf(wb[4 * k + 2], u.z, c0); c0 = fmaf(wb[4 * k + 3], u.w, c0);
                    a1 = fmaf(wa[4 * k], v.x, a1); a1 = fmaf(wa[4 * k + 1], v.y, a1);
                    a1 = fmaf(wa[4 * k + 2], v.z, a1); a1 = fmaf(wa[4 * k + 3], v.w, a1);
                    c1 = fmaf(wb[4 * k], v.x, c1); c1 = fmaf(wb[4 * k + 1], v.y, c1);
                    c1 = fmaf(wb[4 * k + 2], v.z, c1); c1 = fmaf(wb[4 * k + 3], v.w, c1);
                }
                const float acc[2][2] = {{a0, c0}, {a1, c1}};
                const int rr[2] = {r0, r1};
#pragma unroll
                for (int q = 0; q < 2; ++q) {
                    if (p + q >= c) break;
                    const int64_t slot = sorted_row[row0 + rr[q]];
#pragma unroll
                    for (int hcol = 0; hcol < 2; ++hcol) {
                        const float a = apply_act(acc[q][hcol], act);
                        const T hi = from_f32<T>(a);
                        h1[slot * d + j + hcol * dh] = hi;
                        if (h1_lo) h1_lo[slot * d + j + hcol * dh] = from_f32<T>(a - to_f32<T>(hi));
                    }
                }
            }
        }
    }
}

// ------------------------------------------------------------------------------------------------
// a2: LayerNorm (L156; A8: biased variance, eps, affine).  One warp per row, fp32 statistics,
// two passes over registers (mean, then centred second moment).
// ------------------------------------------------------------------------------------------------
template <typename T, int D>
__global__ void __launch_bounds__(256)
k_layernorm(const float* __restrict__ h, int N, const float* __restrict__ gamma,
            const float* __restrict__ beta, float eps, T* __restrict__ u, T* __restrict__ u_lo) {
    constexpr int PER = D / 32;
    int row = blockIdx.x * 8 + (threadIdx.x >> 5);
    int lane = threadIdx.x & 31;
    if (row >= N) return;
    const float* hp = h + (int64_t)row * D;
    float v[PER];
    float s = 0.f;
#pragma unroll
    for (int i = 0; i < PER; ++i) { v[i] = hp[lane + 32 * i]; s += v[i]; }
    float mean = warp_sum(s) * (1.0f / D);
    float q = 0.f;
#pragma unroll
    for (int i = 0; i < PER; ++i) { float c = v[i] - mean; q = fmaf(c, c, q); }
    float rstd = rsqrtf(warp_sum(q) * (1.0f / D) + eps);
    T* up = u + (int64_t)row * D;
#pragma unroll
    for (int i = 0; i < PER; ++i) {
        int c = lane + 32 * i;
        const float y = (v[i] - mean) * rstd * gamma[c] + beta[c];
        const T hi = from_f32<T>(y);
        up[c] = hi;
        if (u_lo) u_lo[(int64_t)row * D + c] = from_f32<T>(y - to_f32<T>(hi));
    }
}

// a2, vectorised: lane owns PER = D / 32 CONTIGUOUS columns (D in {64, 128, 256, 512}), 128-bit loads of h / gamma /
// beta and 64/128-bit stores of the bf16 outputs; same arithmetic (fp32 statistics, two passes over registers).
template <int D>
__global__ void __launch_bounds__(256)
k_layernorm_vec(const float* __restrict__ h, int N, const float* __restrict__ gamma, const float* __restrict__ beta,
                float eps, bf16* __restrict__ u, bf16* __restrict__ u_lo, uint8_t* __restrict__ u8, float u8_scale) {
    constexpr int PER = D / 32, V = PER < 4 ? PER : 4;            // floats per vector load
    const int row = blockIdx.x * 8 + (threadIdx.x >> 5), lane = threadIdx.x & 31;
    if (row >= N) return;
    const float* hp = h + (int64_t)row * D + lane * PER;
    float v[PER], g[PER], b[PER];
#pragma unroll
    for (int i = 0; i < PER; i += V) {
        if (V == 4) {
            *reinterpret_cast<float4*>(&v[i]) = *reinterpret_cast<const float4*>(hp + i);
            *reinterpret_cast<float4*>(&g[i]) = __ldg(reinterpret_cast<const float4*>(gamma + lane * PER + i));
            *reinterpret_cast<float4*>(&b[i]) = __ldg(reinterpret_cast<const float4*>(beta + lane * PER + i));
        } else {
            *reinterpret_cast<float2*>(&v[i]) = *reinterpret_cast<const float2*>(hp + i);
            *reinterpret_cast<float2*>(&g[i]) = __ldg(reinterpret_cast<const float2*>(gamma + lane * PER + i));
            *reinterpret_cast<float2*>(&b[i]) = __ldg(reinterpret_cast<const float2*>(beta + lane * PER + i));
        }
    }
    float s = 0.f;
#pragma unroll
    for (int i = 0; i < PER; ++i) s += v[i];
    const float mean = warp_sum(s) * (1.0f / D);
    float q = 0.f;
#pragma unroll
    for (int i = 0; i < PER; ++i) { const float c = v[i] - mean; q = fmaf(c, c, q); }
    const float rstd = rsqrtf(warp_sum(q) * (1.0f / D) + eps);
    uint32_t hi[PER / 2], lo[PER / 2];
    uint16_t q8[PER / 2];
#pragma unroll
    for (int i = 0; i < PER / 2; ++i) {
        const float y0 = (v[2 * i] - mean) * rstd * g[2 * i] + b[2 * i];
        const float y1 = (v[2 * i + 1] - mean) * rstd * g[2 * i + 1] + b[2 * i + 1];
        q8[i] = (uint16_t)__nv_cvt_float2_to_fp8x2(make_float2(y0 * u8_scale, y1 * u8_scale), __NV_SATFINITE, __NV_E4M3);
        __nv_bfloat162 h2 = __floats2bfloat162_rn(y0, y1);
        hi[i] = *reinterpret_cast<uint32_t*>(&h2);
        __nv_bfloat162 l2 = __floats2bfloat162_rn(y0 - __low2float(h2), y1 - __high2float(h2));
        lo[i] = *reinterpret_cast<uint32_t*>(&l2);
    }
    const int64_t o = (int64_t)row * D + lane * PER;
    auto store = [&](bf16* dst, const uint32_t (&w)[PER / 2]) {
        if (PER >= 8) {
#pragma unroll
            for (int i = 0; i < PER / 8; ++i)
                reinterpret_cast<uint4*>(dst + o)[i] = make_uint4(w[4 * i], w[4 * i + 1], w[4 * i + 2], w[4 * i + 3]);
        } else if (PER == 4) {
            *reinterpret_cast<uint2*>(dst + o) = make_uint2(w[0], w[1]);
        } else {
            *reinterpret_cast<uint32_t*>(dst + o) = w[0];
        }
    };
    store(u, hi);
    if (u_lo) store(u_lo, lo);
    if (u8) {                                                     // e4m3 copy (NEXT-3: FP8 operands of the QKV projection)
#pragma unroll
        for (int i = 0; i < PER / 2; ++i) reinterpret_cast<uint16_t*>(u8 + (int64_t)row * D + lane * PER)[i] = q8[i];
    }
}

// ------------------------------------------------------------------------------------------------
// CUDA-core GEMM  C = A[M,K] W[N,K]^T with the shared epilogue (fp32 debug path / debugging aid).
// 64x64 tile, BK = 16, 256 threads x (4x4) outputs, fp32 accumulate.  K % 16 == 0, N % 64 == 0.
// ------------------------------------------------------------------------------------------------
template <typename T>
__global__ void __launch_bounds__(256)
k_gemm_simple(const T* __restrict__ A, const T* __restrict__ A_lo, const T* __restrict__ W, int M, int N, int K, Epi ep) {
    __shared__ float As[16][64 + 4];
    __shared__ float Ws[16][64 + 4];
    const int m0 = blockIdx.y * 64, n0 = blockIdx.x * 64;
    int64_t w_row0 = 0;
    if (ep.group_offsets) {
        int g = 1;
        if (m0 >= ep.group_offsets[ep.n_groups + 1]) return;
        while (g < ep.n_groups && m0 >= ep.group_offsets[g + 1]) ++g;
        w_row0 = (int64_t)(g - 1) * N;
    } else if (ep.group_rows > 0) w_row0 = (int64_t)(m0 / ep.group_rows) * N;
    const int tx = threadIdx.x & 15, ty = threadIdx.x >> 4;
    float acc[4][4] = {};
    const int lr = threadIdx.x >> 2, lk = (threadIdx.x & 3) * 4;   // 64 rows x 16 k, 4 k per thread
    for (int k0 = 0; k0 < K; k0 += 16) {
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            int m = m0 + lr;
            float a = (m < M) ? to_f32<T>(A[(int64_t)m * K + k0 + lk + i]) : 0.0f;
            if (A_lo && m < M) a += to_f32<T>(A_lo[(int64_t)m * K + k0 + lk + i]);
            As[lk + i][lr] = a;
            Ws[lk + i][lr] = to_f32<T>(W[(w_row0 + n0 + lr) * K + k0 + lk + i]);
        }
        __syncthreads();
#pragma unroll
        for (int k = 0; k < 16; ++k) {
            float a[4], b[4];
#pragma unroll
            for (int i = 0; i < 4; ++i) { a[i] = As[k][ty * 4 + i]; b[i] = Ws[k][tx * 4 + i]; }
#pragma unroll
            for (int i = 0; i < 4; ++i)
#pragma unroll
                for (int j = 0; j < 4; ++j) acc[i][j] = fmaf(a[i], b[j], acc[i][j]);
        }
        __syncthreads();
    }
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        int m = m0 + ty * 4 + i;
        if (m >= M) continue;
        int row = ep.row_perm ? ep.row_perm[m] : m;
        if (row < 0) continue;
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            int n = n0 + tx * 4 + j;
            float v = acc[i][j];
            if (ep.bias) v += ep.bias[w_row0 + n];
            v = apply_act(v, ep.act);
            if (ep.residual) v += ep.residual[(int64_t)row * ep.ld_res + n];
            if (ep.out_f32) ep.out_f32[(int64_t)row * ep.ld_f32 + n] = v;
            if (ep.out_act) {
                const T hi = from_f32<T>(v);
                ((T*)ep.out_act)[(int64_t)row * ep.ld_act + n] = hi;
                if (ep.out_act_lo) ((T*)ep.out_act_lo)[(int64_t)row * ep.ld_act + n] = from_f32<T>(v - to_f32<T>(hi));
            }
        }
    }
}

// ------------------------------------------------------------------------------------------------
// a4 (debug path): per event, per head  O = softmax(Q K^T / sqrt(hd)) V  (Eq. 4) with the
// FlashAttention recurrence (L154) over key tiles of 32; one thread per query row, fp32 state.
// Keys outside the event or with valid == 0 get weight exactly 0 (A2); no valid key -> O = 0 (A15).
// grid = (n_tiles, H), block = tile_q threads; work = (event, q_tile) list.
// ------------------------------------------------------------------------------------------------
template <typename T, int HD>
__global__ void __launch_bounds__(128)
k_attn_simple(const T* __restrict__ QKV, const int* __restrict__ key_valid, const int* __restrict__ offsets,
              const int2* __restrict__ work, int tile_q, int d, T* __restrict__ O, T* __restrict__ O_lo) {
    __shared__ float Ks[32][HD + 1];
    __shared__ float Vs[32][HD + 1];
    __shared__ int vs[32];
    const int2 wk = work[blockIdx.x];
    const int head = blockIdx.y;
    const int ev0 = offsets[wk.x], ev1 = offsets[wk.x + 1];
    const int qrow = ev0 + wk.y * tile_q + threadIdx.x;
    const bool active = (int)threadIdx.x < tile_q && qrow < ev1;
    const float scale = rsqrtf((float)HD);
    float q[HD], acc[HD];
#pragma unroll
    for (int c = 0; c < HD; ++c) {
        q[c] = active ? to_f32<T>(QKV[(int64_t)qrow * (3 * d) + head * HD + c]) * scale : 0.0f;
        acc[c] = 0.0f;
    }
    float m = -INFINITY, l = 0.0f;
    for (int k0 = ev0; k0 < ev1; k0 += 32) {
        __syncthreads();
        for (int idx = threadIdx.x; idx < 32 * HD; idx += blockDim.x) {
            int j = idx / HD, c = idx % HD;          // K rows: contiguous over c
            int key = k0 + j;
            Ks[j][c] = (key < ev1) ? to_f32<T>(QKV[(int64_t)key * (3 * d) + d + head * HD + c]) : 0.0f;
        }
        for (int idx = threadIdx.x; idx < 32 * HD; idx += blockDim.x) {
            int j = idx / HD, c = idx % HD;
            int key = k0 + j;
            Vs[j][c] = (key < ev1) ? to_f32<T>(QKV[(int64_t)key * (3 * d) + 2 * d + head * HD + c]) : 0.0f;
        }
        if (threadIdx.x < 32) {
            int key = k0 + threadIdx.x;
            vs[threadIdx.x] = (key < ev1) && (key_valid == nullptr || key_valid[key] != 0);
        }
        __syncthreads();
        float s[32];
        float tmax = -INFINITY;
#pragma unroll
        for (int j = 0; j < 32; ++j) {
            float a = 0.0f;
#pragma unroll
            for (int c = 0; c < HD; ++c) a = fmaf(q[c], Ks[j][c], a);
            s[j] = vs[j] ? a : -INFINITY;
            tmax = fmaxf(tmax, s[j]);
        }
        if (tmax == -INFINITY) continue;             // block-uniform only per thread; no barrier inside
        float mnew = fmaxf(m, tmax);
        float corr = expf(m - mnew);                 // m = -inf -> 0
        l *= corr;
#pragma unroll
        for (int c = 0; c < HD; ++c) acc[c] *= corr;
#pragma unroll
        for (int j = 0; j < 32; ++j) {
            float p = expf(s[j] - mnew);             // -inf -> 0
            l += p;
#pragma unroll
            for (int c = 0; c < HD; ++c) acc[c] = fmaf(p, Vs[j][c], acc[c]);
        }
        m = mnew;
    }
    if (active) {
        float inv = (l > 0.0f) ? 1.0f / l : 0.0f;
#pragma unroll
        for (int c = 0; c < HD; ++c) {
            const float y = acc[c] * inv;
            const T hi = from_f32<T>(y);
            O[(int64_t)qrow * d + head * HD + c] = hi;
            if (O_lo) O_lo[(int64_t)qrow * d + head * HD + c] = from_f32<T>(y - to_f32<T>(hi));
        }
    }
}

// ------------------------------------------------------------------------------------------------
// a8 (output layer): out[row, o] = W2[o,:] . hidden[row, head(o) block] + b2[o] in fp32; one warp per
// row; rows with valid == 0 are written as exactly 0 (A2).  hidden = [N, n_blocks*d]; output o reads
// hidden block blk[o].  Outputs 0..C-1 -> logits, C.. -> regress.
// ------------------------------------------------------------------------------------------------

// output o of a row: [binary (n_bin = 0 | 1)] [class logits (n_cls)] [regressions (n_reg)]  (L156 / Fig. 2)
__device__ __forceinline__ void heads_store(const HeadsOut& ho, int row, int o, float a, float* __restrict__ out_logits,
                                            float* __restrict__ out_regress, float* __restrict__ out_binary) {
    if (o < ho.n_bin) { if (out_binary) out_binary[row] = a; }
    else if (o < ho.n_bin + ho.n_cls) out_logits[(int64_t)row * ho.n_cls + (o - ho.n_bin)] = a;
    else out_regress[(int64_t)row * ho.n_reg + (o - ho.n_bin - ho.n_cls)] = a;
}

template <typename T>
__global__ void __launch_bounds__(256)
k_heads_l2(const T* __restrict__ hidden, const T* __restrict__ hidden_lo, int N, int d, int ld_hidden, const float* __restrict__ W2,
           const float* __restrict__ b2, const int* __restrict__ valid, const int* __restrict__ hid_row, HeadsOut ho,
           float* __restrict__ out_logits, float* __restrict__ out_regress, float* __restrict__ out_binary) {
    int row = blockIdx.x * 8 + (threadIdx.x >> 5);
    int lane = threadIdx.x & 31;
    if (row >= N) return;
    const int hrow = hid_row ? hid_row[row] : (valid[row] != 0 ? row : -1);   // row of `hidden` holding this element (-1: pad row)
    const bool ok = hrow >= 0;
    const T* hp = hidden + (int64_t)(ok ? hrow : 0) * ld_hidden;
    for (int o = 0; o < ho.n_out; ++o) {
        float a = 0.0f;
        if (ok) {
            const T* hb = hp + ho.blk[o] * d;
            const float* w = W2 + (int64_t)o * d;
            if (hidden_lo) {
                const T* lb = hidden_lo + (int64_t)hrow * ld_hidden + ho.blk[o] * d;
                for (int c = lane; c < d; c += 32) a = fmaf(to_f32<T>(hb[c]) + to_f32<T>(lb[c]), w[c], a);
            } else {
                for (int c = lane; c < d; c += 32) a = fmaf(to_f32<T>(hb[c]), w[c], a);
            }
            a = warp_sum(a) + b2[o];
        }
        if (lane == 0) heads_store(ho, row, o, a, out_logits, out_regress, out_binary);
    }
}

// a8 output layer, bf16 path: the same computation with 128-bit loads (lane = 8 consecutive hidden units per 256-wide
// chunk, d <= 512, at most 5 head blocks): all of the row's hidden vectors (hi + lo) are requested up front (one
// round trip to HBM), then each is reused by all outputs of its block.
template <int NCH>
__global__ void __launch_bounds__(256)
k_heads_l2_vec(const bf16* __restrict__ hidden, const bf16* __restrict__ hidden_lo, int N, int d, int ld_hidden, int n_blk,
               const float* __restrict__ W2, const float* __restrict__ b2, const int* __restrict__ valid, const int* __restrict__ hid_row, HeadsOut ho,
               float* __restrict__ out_logits, float* __restrict__ out_regress, float* __restrict__ out_binary) {
    const int row = blockIdx.x * 8 + (threadIdx.x >> 5);
    const int lane = threadIdx.x & 31;
    if (row >= N) return;
    const int hrow = hid_row ? hid_row[row] : (valid[row] != 0 ? row : -1);
    const bool ok = hrow >= 0;
    uint4 hraw[MAX_HBLK][NCH], lraw[MAX_HBLK][NCH];
#pragma unroll
    for (int b = 0; b < MAX_HBLK; ++b)
#pragma unroll
        for (int ch = 0; ch < NCH; ++ch) {
            const int c = ch * 256 + lane * 8;
            hraw[b][ch] = make_uint4(0, 0, 0, 0); lraw[b][ch] = make_uint4(0, 0, 0, 0);
            if (ok && b < n_blk && c < d) {
                const int64_t off = (int64_t)hrow * ld_hidden + b * d + c;
                hraw[b][ch] = *reinterpret_cast<const uint4*>(hidden + off);
                if (hidden_lo) lraw[b][ch] = *reinterpret_cast<const uint4*>(hidden_lo + off);
            }
        }
    for (int o = 0; o < ho.n_out; ++o) {
        float a = 0.0f;
        if (ok) {
            const int b = ho.blk[o];
#pragma unroll
            for (int ch = 0; ch < NCH; ++ch) {
                const int c = ch * 256 + lane * 8;
                if (c < d) {
                    uint4 h4 = hraw[0][ch], l4 = lraw[0][ch];
#pragma unroll
                    for (int bb = 1; bb < MAX_HBLK; ++bb) if (b == bb) { h4 = hraw[bb][ch]; l4 = lraw[bb][ch]; }
                    const uint32_t hw[4] = {h4.x, h4.y, h4.z, h4.w}, lw[4] = {l4.x, l4.y, l4.z, l4.w};
                    const float4* wp = reinterpret_cast<const float4*>(W2 + (int64_t)o * d + c);
                    const float4 w0 = __ldg(wp), w1 = __ldg(wp + 1);
                    const float wv[8] = {w0.x, w0.y, w0.z, w0.w, w1.x, w1.y, w1.z, w1.w};
#pragma unroll
                    for (int i = 0; i < 4; ++i) {
                        a = fmaf(__uint_as_float(hw[i] << 16) + __uint_as_float(lw[i] << 16), wv[2 * i], a);
                        a = fmaf(__uint_as_float(hw[i] & 0xffff0000u) + __uint_as_float(lw[i] & 0xffff0000u), wv[2 * i + 1], a);
                    }
                }
            }
            a = warp_sum(a) + b2[o];
        }
        if (lane == 0) heads_store(ho, row, o, a, out_logits, out_regress, out_binary);
    }
}

// a8 output layer, bf16 path, at most 16 outputs: as k_heads_l2_vec, but every hidden vector is unpacked (hi + lo) once,
// the head block of an output is chosen by a warp-uniform switch over statically indexed registers (no per-output
// select chains), and the 16 per-lane partial sums are reduced together by a halving butterfly (16 shuffles instead
// of 5 per output; the additions happen in the same order as warp_sum's, so the results are bit-identical to
// k_heads_l2_vec's).  After the butterfly lane 2o holds output o.
template <int HALF>
__device__ __forceinline__ void heads_fold(float (&acc)[16], int lane) {
    constexpr int BIT = HALF * 2;
    const bool up = (lane & BIT) != 0;
#pragma unroll
    for (int j = 0; j < HALF; ++j) {
        const float mine = up ? acc[j + HALF] : acc[j];
        const float other = up ? acc[j] : acc[j + HALF];
        acc[j] = mine + __shfl_xor_sync(0xffffffffu, other, BIT);
    }
}
__device__ __forceinline__ float heads_dot8(const float (&h)[8], const float4& w0, const float4& w1, float a) {
    a = fmaf(h[0], w0.x, a); a = fmaf(h[1], w0.y, a); a = fmaf(h[2], w0.z, a); a = fmaf(h[3], w0.w, a);
    a = fmaf(h[4], w1.x, a); a = fmaf(h[5], w1.y, a); a = fmaf(h[6], w1.z, a); a = fmaf(h[7], w1.w, a);
    return a;
}
template <int NCH>
__global__ void __launch_bounds__(256)
k_heads_l2_fold(const bf16* __restrict__ hidden, const bf16* __restrict__ hidden_lo, int N, int d, int ld_hidden, int n_blk,
                const float* __restrict__ W2, const float* __restrict__ b2, const int* __restrict__ valid, const int* __restrict__ hid_row, HeadsOut ho,
                float* __restrict__ out_logits, float* __restrict__ out_regress, float* __restrict__ out_binary) {
    const int row = blockIdx.x * 8 + (threadIdx.x >> 5);
    const int lane = threadIdx.x & 31;
    if (row >= N) return;
    const int hrow = hid_row ? hid_row[row] : (valid[row] != 0 ? row : -1);   // warp-uniform
    const bool ok = hrow >= 0;
    float acc[16];
#pragma unroll
    for (int o = 0; o < 16; ++o) acc[o] = 0.0f;
    if (ok) {
        float hv[MAX_HBLK][NCH][8];
#pragma unroll
        for (int b = 0; b < MAX_HBLK; ++b)
#pragma unroll
            for (int ch = 0; ch < NCH; ++ch) {
                const int c = ch * 256 + lane * 8;
                uint4 h4 = make_uint4(0, 0, 0, 0), l4 = make_uint4(0, 0, 0, 0);
                if (b < n_blk && c < d) {
                    const int64_t off = (int64_t)hrow * ld_hidden + b * d + c;
                    h4 = *reinterpret_cast<const uint4*>(hidden + off);
                    if (hidden_lo) l4 = *reinterpret_cast<const uint4*>(hidden_lo + off);
                }
                const uint32_t hw[4] = {h4.x, h4.y, h4.z, h4.w}, lw[4] = {l4.x, l4.y, l4.z, l4.w};
#pragma unroll
                for (int i = 0; i < 4; ++i) {
                    hv[b][ch][2 * i] = __uint_as_float(hw[i] << 16) + __uint_as_float(lw[i] << 16);
                    hv[b][ch][2 * i + 1] = __uint_as_float(hw[i] & 0xffff0000u) + __uint_as_float(lw[i] & 0xffff0000u);
                }
            }
#pragma unroll
        for (int o = 0; o < 16; ++o) {
            if (o < ho.n_out) {
                const int b = ho.blk[o];
#pragma unroll
                for (int ch = 0; ch < NCH; ++ch) {
                    const int c = ch * 256 + lane * 8;
                    if (c < d) {
                        const float4* wp = reinterpret_cast<const float4*>(W2 + (int64_t)o * d + c);
                        const float4 w0 = __ldg(wp), w1 = __ldg(wp + 1);
                        switch (b) {
                            case 0: acc[o] = heads_dot8(hv[0][ch], w0, w1, acc[o]); break;
                            case 1: acc[o] = heads_dot8(hv[1][ch], w0, w1, acc[o]); break;
                            case 2: acc[o] = heads_dot8(hv[2][ch], w0, w1, acc[o]); break;
                            case 3: acc[o] = heads_dot8(hv[3][ch], w0, w1, acc[o]); break;
                            case 4: acc[o] = heads_dot8(hv[4][ch], w0, w1, acc[o]); break;
                            default: acc[o] = heads_dot8(hv[5][ch], w0, w1, acc[o]); break;
                        }
                    }
                }
            }
        }
        heads_fold<8>(acc, lane);
        heads_fold<4>(acc, lane);
        heads_fold<2>(acc, lane);
        heads_fold<1>(acc, lane);
        acc[0] += __shfl_xor_sync(0xffffffffu, acc[0], 1);
    }
    const int o = lane >> 1;
    if ((lane & 1) == 0 && o < ho.n_out) {
        const float a = ok ? acc[0] + b2[o] : 0.0f;
        heads_store(ho, row, o, a, out_logits, out_regress, out_binary);
    }
}

// int 0/1 per row -> one bit per row (kernel-level attention entry; the model path gets the bits from k_sched_count)
__global__ void k_pack_valid_bits(const int* __restrict__ valid, int N, uint32_t* __restrict__ bits) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const unsigned vb = __ballot_sync(0xffffffffu, i < N && valid[i] != 0);
    if ((threadIdx.x & 31) == 0) bits[i >> 5] = vb;
}
void launch_pack_valid_bits(const int* valid, int N, uint32_t* bits, cudaStream_t st) {
    k_pack_valid_bits<<<(N + 255) / 256, 256, 0, st>>>(valid, N, bits);
}

// final_ln = 0 (reading A7 off): the heads read the residual stream itself, u = T(h) (+ u_lo = T(h - u))
template <typename T>
__global__ void k_cast_rows(const float* __restrict__ h, int64_t n, T* __restrict__ u, T* __restrict__ u_lo) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const float v = h[i];
    const T hi = from_f32<T>(v);
    u[i] = hi;
    if (u_lo) u_lo[i] = from_f32<T>(v - to_f32<T>(hi));
}
void launch_cast_rows(bool fp32, const float* h, int64_t n, void* u, void* u_lo, cudaStream_t st) {
    const unsigned grid = (unsigned)((n + 255) / 256);
    if (fp32) k_cast_rows<float><<<grid, 256, 0, st>>>(h, n, (float*)u, (float*)u_lo);
    else k_cast_rows<bf16><<<grid, 256, 0, st>>>(h, n, (bf16*)u, (bf16*)u_lo);
}

// fp32 <- T conversion for the debug taps
template <typename T>
__global__ void k_to_f32(const T* __restrict__ src, float* __restrict__ dst, int64_t n) {
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) dst[i] = to_f32<T>(src[i]);
}

// debug tap: rows of a compacted [Nc, cols] matrix back to their original rows (pad rows -> 0)
__global__ void k_uncompact(const float* __restrict__ src, const int* __restrict__ comp_row, float* __restrict__ out, int64_t N, int cols) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N * cols) return;
    const int c = comp_row[i / cols];
    out[i] = c >= 0 ? src[(int64_t)c * cols + i % cols] : 0.0f;
}
void launch_uncompact(const float* src, const int* comp_row, float* out, int64_t N, int cols, cudaStream_t st) {
    k_uncompact<<<(unsigned)((N * cols + 255) / 256), 256, 0, st>>>(src, comp_row, out, N, cols);
}

// debug tap: the fused blocks' tiled residual-stream layout (tc_post.cu h_off) -> row-major
__global__ void k_untile_h(const float* __restrict__ ht, float* __restrict__ out, int64_t N, int d) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N * d) return;
    const int64_t row = i / d; const int col = (int)(i % d);
    out[i] = ht[(row / 128) * (128 * (int64_t)d) + (col >> 2) * 512 + (row % 128) * 4 + (col & 3)];
}
void launch_untile_h(const float* ht, float* out, int64_t N, int d, cudaStream_t st) {
    k_untile_h<<<(unsigned)((N * d + 255) / 256), 256, 0, st>>>(ht, out, N, d);
}

// Two parallel encoders run as ONE batch over 2 N_pad rows: stack g owns rows [g N_pad, g N_pad + N)
// (N_pad = N rounded up to 128) and the virtual events g (E + 1) .. g (E + 1) + E - 1; virtual event g (E + 1) + E is the
// gap [g N_pad + N, (g + 1) N_pad), which no work item touches.  This kernel copies the schedule arrays the per-row
// kernels read (and the embedded residual stream) from stack 0's rows to stack g's (g >= 1).
__global__ void k_sched_replicate(int N, int N_pad, int E, int g, int d, int* __restrict__ offsets, int* __restrict__ n_valid,
                                  int* __restrict__ row_event, int* __restrict__ valid, uint32_t* __restrict__ valid_bits,
                                  float* __restrict__ h) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int64_t base = (int64_t)g * N_pad;
    const int Ev = E + 1;
    if (i < N) { row_event[base + i] = row_event[i] + g * Ev; valid[base + i] = valid[i]; }
    if (i < N_pad - N) { row_event[base - N_pad + N + i] = (g - 1) * Ev + E; valid[base - N_pad + N + i] = 0; }   // the gap before this stack
    if (i < N_pad / 32) valid_bits[base / 32 + i] = (i * 32 < N) ? valid_bits[i] : 0u;
    if (i < E) n_valid[g * Ev + i] = n_valid[i];
    if (i <= E) offsets[g * Ev + i] = (int)base + offsets[i];
    if (i == 0) { offsets[(g + 1) * Ev] = (int)base + N_pad; n_valid[g * Ev + E] = 0; n_valid[(g - 1) * Ev + E] = 0; }
    if (i < (int64_t)N * d / 4) reinterpret_cast<float4*>(h + base * d)[i] = reinterpret_cast<const float4*>(h)[i];
}
void launch_sched_replicate(int N, int N_pad, int E, int g, int d, int* offsets, int* n_valid, int* row_event, int* valid,
                            uint32_t* valid_bits, float* h, cudaStream_t st) {
    const int64_t n = (int64_t)N * d / 4;
    k_sched_replicate<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(N, N_pad, E, g, d, offsets, n_valid, row_event, valid, valid_bits, h);
}

// ------------------------------------------------------------------------------------------------ micro-benchmarks
// Throughput of the units that bound the attention softmax (bench.py's roofline.alu object): results per clock per SM of
//   0: ex2.approx.ftz.f32 (MUFU)   1: ex2.approx.ftz.bf16x2 (MUFU, two results per instruction)
//   2: the Cody-Waite + degree-3 polynomial 2^x on packed fp32 pairs (FMA / ALU pipes), as tc_attn2.cu uses it
//   3: fma.rn.f32x2 (packed FMA)
// One CTA of 1024 threads per SM, 8 independent dependency chains per thread, cycles from clock64 around the loop.
__global__ void __launch_bounds__(1024, 1)
k_microbench(int which, int iters, float seed, float* __restrict__ per_block, float* __restrict__ sink) {
    float v[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) v[i] = seed - 0.01f * (float)(threadIdx.x & 7) - 0.001f * (float)i;
    __syncthreads();
    const long long t0 = clock64();
    if (which == 0) {
        for (int it = 0; it < iters; ++it) {
#pragma unroll
            for (int i = 0; i < 8; ++i) asm volatile("ex2.approx.ftz.f32 %0, %0;" : "+f"(v[i]));
        }
    } else if (which == 1) {
        uint32_t u[8];
#pragma unroll
        for (int i = 0; i < 8; ++i) u[i] = 0xbf00be80u + (uint32_t)i;                  // pairs of small negative bf16
        for (int it = 0; it < iters; ++it) {
#pragma unroll
            for (int i = 0; i < 8; ++i) asm volatile("ex2.approx.ftz.bf16x2 %0, %0;" : "+r"(u[i]));
        }
#pragma unroll
        for (int i = 0; i < 8; ++i) v[i] = __uint_as_float(u[i]);
    } else if (which == 2) {
        for (int it = 0; it < iters; ++it) {
#pragma unroll
            for (int i = 0; i < 8; i += 2) {
                float xr0 = fmaf(v[i], 0.2550348616f, 12582912.0f - 8.0f), xr1 = fmaf(v[i + 1], 0.2550348616f, 12582912.0f - 8.0f);
                const float m0 = xr0 - (12582912.0f - 8.0f), m1 = xr1 - (12582912.0f - 8.0f);
                const float f0 = fmaf(v[i], 0.2550348616f, -m0), f1 = fmaf(v[i + 1], 0.2550348616f, -m1);
                float p0 = fmaf(f0, 0.0550089306f, 0.2422109596f), p1 = fmaf(f1, 0.0550089306f, 0.2422109596f);
                p0 = fmaf(p0, f0, 0.6932829272f); p1 = fmaf(p1, f1, 0.6932829272f);
                p0 = fmaf(p0, f0, 1.0f); p1 = fmaf(p1, f1, 1.0f);
                v[i] = __int_as_float(__float_as_int(p0) + (__float_as_int(xr0) << 23)) - 1.0f;   // keeps the chain's argument <= 0
                v[i + 1] = __int_as_float(__float_as_int(p1) + (__float_as_int(xr1) << 23)) - 1.0f;
            }
        }
    } else {
        for (int it = 0; it < iters; ++it) {
#pragma unroll
            for (int i = 0; i < 8; i += 2)
                asm volatile("{\n\t.reg .b64 a, b;\n\tmov.b64 a, {%0, %1};\n\tmov.b64 b, {%2, %2};\n\tfma.rn.f32x2 a, a, b, b;\n\tmov.b64 {%0, %1}, a;\n\t}"
                             : "+f"(v[i]), "+f"(v[i + 1]) : "f"(0.999f));
        }
    }
    const long long t1 = clock64();
    float acc = 0.f;
#pragma unroll
    for (int i = 0; i < 8; ++i) acc += v[i];
    if (acc == 123.456f) sink[0] = acc;
    __shared__ long long tmin, tmax;
    if (threadIdx.x == 0) { tmin = t0; tmax = t1; }
    __syncthreads();
    atomicMin(&tmin, t0); atomicMax(&tmax, t1);
    __syncthreads();
    if (threadIdx.x == 0) per_block[blockIdx.x] = (float)(tmax - tmin);
}
// returns results per clock per SM (mean over one CTA per SM), < 0 on a CUDA error
float launch_microbench(int which, int iters, int num_sms, cudaStream_t st) {
    float *d_cyc = nullptr, *d_sink = nullptr;
    if (cudaMalloc(&d_cyc, num_sms * 4) != cudaSuccess || cudaMalloc(&d_sink, 4) != cudaSuccess) { cudaFree(d_cyc); return -1.0f; }
    k_microbench<<<num_sms, 1024, 0, st>>>(which, iters, -0.5f, d_cyc, d_sink);      // warm-up
    k_microbench<<<num_sms, 1024, 0, st>>>(which, iters, -0.5f, d_cyc, d_sink);
    std::vector<float> cyc(num_sms);
    cudaError_t e = cudaMemcpyAsync(cyc.data(), d_cyc, num_sms * 4, cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    cudaFree(d_cyc); cudaFree(d_sink);
    if (e != cudaSuccess) return -1.0f;
    double mean = 0.0;
    for (float c : cyc) mean += c;
    mean /= num_sms;
    const double per_op = (which == 1) ? 2.0 : 1.0;          // bf16x2: two results per instruction; fma.f32x2 pairs are counted as issued above
    return (float)(1024.0 * iters * 8.0 * per_op / mean);
}

// ------------------------------------------------------------------------------------------------ launchers
int launch_schedule(const float* X, int N, int F, const int* offsets, int E, int* block_counts, int* block_base,
                    int* valid, uint32_t* valid_bits, int* row_event, int* row_pos, int* n_valid, int* type_offsets, int* sorted_row,
                    int* type_perm, const SchedCompact& sc, cudaStream_t st) {
    const int nb = (N + SCHED_BLOCK - 1) / SCHED_BLOCK;
    k_sched_count<<<nb, SCHED_BLOCK, 0, st>>>(X, N, F, offsets, E, block_counts, valid, valid_bits, row_event, row_pos, n_valid);
    k_sched_scan<<<1, 32, 0, st>>>(block_counts, nb, block_base, type_offsets, sc.block_vbase, sc.n_comp);
    k_sched_scatter<<<nb, SCHED_BLOCK, 0, st>>>(X, N, F, block_base, type_offsets, sc.block_vbase, row_event, sorted_row, type_perm,
                                                sc.vbefore, sc.comp_row, sc.orig_row, sc.row_event_c, sc.comp_type_perm);
    k_sched_offsets_c<<<1, 256, 0, st>>>(offsets, E, N, sc.vbefore, sc.n_comp, sc.offsets_c);
    return 4;
}

// a1 on the tensor pipe, step 1: the fp32 features of every non-pad row as bf16 terms in its type-sorted slot,
//   xa[slot] = [x_hi | x_lo | x_hi]  (3 x 64 columns, features padded with zeros to 64),  x_hi = T(x), x_lo = T(x - x_hi),
// so that ONE K = 192 GEMM against [W_hi | W_hi | W_lo] (built in mlpf_create) gives x W^T to ~2^-17 relative (the x_lo W_lo
// term is dropped): the first embedding layer keeps its fp32 weights' precision (reading A3) on the bf16 tensor pipe.
constexpr int PACK_ROWS = 32;
__global__ void __launch_bounds__(256)
k_embed_pack(const float* __restrict__ X, int N, int F, const int* __restrict__ sorted_row, bf16* __restrict__ xa) {
    __shared__ float xs[PACK_ROWS][64];
    __shared__ int slot[PACK_ROWS];
    const int row0 = blockIdx.x * PACK_ROWS;
    const int rows = min(PACK_ROWS, N - row0);
    for (int idx = threadIdx.x; idx < PACK_ROWS * 64; idx += 256) {
        const int r = idx >> 6, k = idx & 63;
        xs[r][k] = (r < rows && k < F) ? X[(int64_t)(row0 + r) * F + k] : 0.0f;
    }
    if (threadIdx.x < PACK_ROWS)
        slot[threadIdx.x] = (threadIdx.x < rows && element_type(X, row0 + threadIdx.x, F) != 0) ? sorted_row[row0 + threadIdx.x] : -1;
    __syncthreads();
    // 24 16-byte pieces per row: piece c = segment c / 8 (hi, lo, hi), features 8 (c % 8) .. + 7
    for (int idx = threadIdx.x; idx < PACK_ROWS * 24; idx += 256) {
        const int r = idx / 24, c = idx % 24;
        const int sl = slot[r];
        if (sl < 0) continue;
        const float* xp = &xs[r][(c & 7) * 8];
        uint32_t w[4];
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            float2 v = make_float2(xp[2 * i], xp[2 * i + 1]);
            __nv_bfloat162 h2 = __floats2bfloat162_rn(v.x, v.y);
            if ((c >> 3) == 1) h2 = __floats2bfloat162_rn(v.x - __low2float(h2), v.y - __high2float(h2));
            w[i] = *reinterpret_cast<uint32_t*>(&h2);
        }
        *reinterpret_cast<uint4*>(xa + (int64_t)sl * 192 + c * 8) = make_uint4(w[0], w[1], w[2], w[3]);
    }
}
void launch_embed_pack(const float* X, int N, int F, const int* sorted_row, void* xa, cudaStream_t st) {
    k_embed_pack<<<(N + PACK_ROWS - 1) / PACK_ROWS, 256, 0, st>>>(X, N, F, sorted_row, (bf16*)xa);
}

void launch_embed_l1(bool fp32, const float* X, int N, int F, int d, const float* W1t, const float* b1, int act,
                     const int* sorted_row, void* h1, void* h1_lo, float* h, cudaStream_t st) {
    dim3 grid((N + EMB_ROWS - 1) / EMB_ROWS);
    if (fp32) k_embed_l1<float><<<grid, EMB_THREADS, 0, st>>>(X, N, F, d, W1t, b1, act, sorted_row, (float*)h1, (float*)h1_lo, h);
    else k_embed_l1<bf16><<<grid, EMB_THREADS, 0, st>>>(X, N, F, d, W1t, b1, act, sorted_row, (bf16*)h1, (bf16*)h1_lo, h);
}

template <typename T>
static int layernorm_d(int d, const float* x, int N, const float* g, const float* b, float eps, T* u, T* u_lo, cudaStream_t st) {
    dim3 grid((N + 7) / 8);
    switch (d) {
        case 64:  k_layernorm<T, 64><<<grid, 256, 0, st>>>(x, N, g, b, eps, u, u_lo); break;
        case 128: k_layernorm<T, 128><<<grid, 256, 0, st>>>(x, N, g, b, eps, u, u_lo); break;
        case 192: k_layernorm<T, 192><<<grid, 256, 0, st>>>(x, N, g, b, eps, u, u_lo); break;
        case 256: k_layernorm<T, 256><<<grid, 256, 0, st>>>(x, N, g, b, eps, u, u_lo); break;
        case 320: k_layernorm<T, 320><<<grid, 256, 0, st>>>(x, N, g, b, eps, u, u_lo); break;
        case 384: k_layernorm<T, 384><<<grid, 256, 0, st>>>(x, N, g, b, eps, u, u_lo); break;
        case 448: k_layernorm<T, 448><<<grid, 256, 0, st>>>(x, N, g, b, eps, u, u_lo); break;
        case 512: k_layernorm<T, 512><<<grid, 256, 0, st>>>(x, N, g, b, eps, u, u_lo); break;
        default: return -1;
    }
    return 0;
}
int launch_layernorm(bool fp32, int d, const float* x, int N, const float* g, const float* b, float eps, void* u,
                     void* u_lo, cudaStream_t st, uint8_t* u8, float u8_scale) {
    if (!fp32) {
        dim3 grid((N + 7) / 8);
        switch (d) {
            case 64:  k_layernorm_vec<64><<<grid, 256, 0, st>>>(x, N, g, b, eps, (bf16*)u, (bf16*)u_lo, u8, u8_scale); return 0;
            case 128: k_layernorm_vec<128><<<grid, 256, 0, st>>>(x, N, g, b, eps, (bf16*)u, (bf16*)u_lo, u8, u8_scale); return 0;
            case 256: k_layernorm_vec<256><<<grid, 256, 0, st>>>(x, N, g, b, eps, (bf16*)u, (bf16*)u_lo, u8, u8_scale); return 0;
            case 512: k_layernorm_vec<512><<<grid, 256, 0, st>>>(x, N, g, b, eps, (bf16*)u, (bf16*)u_lo, u8, u8_scale); return 0;
        }
    }
    return fp32 ? layernorm_d<float>(d, x, N, g, b, eps, (float*)u, (float*)u_lo, st)
                : layernorm_d<bf16>(d, x, N, g, b, eps, (bf16*)u, (bf16*)u_lo, st);
}

void launch_gemm_simple(bool fp32, const void* A, const void* A_lo, const void* W, int M, int N, int K, const Epi& ep,
                        cudaStream_t st) {
    dim3 grid(N / 64, (M + 63) / 64);
    if (fp32) k_gemm_simple<float><<<grid, 256, 0, st>>>((const float*)A, (const float*)A_lo, (const float*)W, M, N, K, ep);
    else k_gemm_simple<bf16><<<grid, 256, 0, st>>>((const bf16*)A, (const bf16*)A_lo, (const bf16*)W, M, N, K, ep);
}

template <typename T>
static void attn_simple_hd(int hd, const T* QKV, const int* key_valid, const int* offsets,
                           const int2* work, int n_tiles, int H, int tile_q, int d, T* O, T* O_lo, cudaStream_t st) {
    dim3 grid((unsigned)n_tiles, H);
    switch (hd) {
        case 16: k_attn_simple<T, 16><<<grid, tile_q, 0, st>>>(QKV, key_valid, offsets, work, tile_q, d, O, O_lo); break;
        case 32: k_attn_simple<T, 32><<<grid, tile_q, 0, st>>>(QKV, key_valid, offsets, work, tile_q, d, O, O_lo); break;
        case 64: k_attn_simple<T, 64><<<grid, tile_q, 0, st>>>(QKV, key_valid, offsets, work, tile_q, d, O, O_lo); break;
    }
}
void launch_attn_simple(bool fp32, int hd, const void* QKV, const int* key_valid,
                        const int* offsets, const int2* work, int n_tiles, int H, int tile_q, int d, void* O,
                        void* O_lo, cudaStream_t st) {
    if (fp32) attn_simple_hd<float>(hd, (const float*)QKV, key_valid, offsets, work, n_tiles, H, tile_q, d, (float*)O, (float*)O_lo, st);
    else attn_simple_hd<bf16>(hd, (const bf16*)QKV, key_valid, offsets, work, n_tiles, H, tile_q, d, (bf16*)O, (bf16*)O_lo, st);
}

void launch_heads_l2(bool fp32, const void* hidden, const void* hidden_lo, int N, int d, int ld_hidden,
                     const float* W2, const float* b2, const int* valid, const int* hid_row, const HeadsOut& ho, float* out_logits,
                     float* out_regress, float* out_binary, cudaStream_t st) {
    dim3 grid((N + 7) / 8);
    if (fp32) k_heads_l2<float><<<grid, 256, 0, st>>>((const float*)hidden, (const float*)hidden_lo, N, d, ld_hidden, W2, b2, valid, hid_row, ho, out_logits, out_regress, out_binary);
    else if (d <= 512 && d % 8 == 0 && ld_hidden % 8 == 0 && ld_hidden / d <= MAX_HBLK) {
        const int n_blk = ld_hidden / d;
        if (ho.n_out <= 16) {
            if (d <= 256) k_heads_l2_fold<1><<<grid, 256, 0, st>>>((const bf16*)hidden, (const bf16*)hidden_lo, N, d, ld_hidden, n_blk, W2, b2, valid, hid_row, ho, out_logits, out_regress, out_binary);
            else k_heads_l2_fold<2><<<grid, 256, 0, st>>>((const bf16*)hidden, (const bf16*)hidden_lo, N, d, ld_hidden, n_blk, W2, b2, valid, hid_row, ho, out_logits, out_regress, out_binary);
        }
        else if (d <= 256) k_heads_l2_vec<1><<<grid, 256, 0, st>>>((const bf16*)hidden, (const bf16*)hidden_lo, N, d, ld_hidden, n_blk, W2, b2, valid, hid_row, ho, out_logits, out_regress, out_binary);
        else k_heads_l2_vec<2><<<grid, 256, 0, st>>>((const bf16*)hidden, (const bf16*)hidden_lo, N, d, ld_hidden, n_blk, W2, b2, valid, hid_row, ho, out_logits, out_regress, out_binary);
    }
    else k_heads_l2<bf16><<<grid, 256, 0, st>>>((const bf16*)hidden, (const bf16*)hidden_lo, N, d, ld_hidden, W2, b2, valid, hid_row, ho, out_logits, out_regress, out_binary);
}

void launch_to_f32(bool fp32, const void* src, float* dst, int64_t n, cudaStream_t st) {
    unsigned grid = (unsigned)((n + 255) / 256);
    if (fp32) k_to_f32<float><<<grid, 256, 0, st>>>((const float*)src, dst, n);
    else k_to_f32<bf16><<<grid, 256, 0, st>>>((const bf16*)src, dst, n);
}

}  // namespace mlpf
