// candidates.cu -- candidate building: the step right after the encoder,
// turning per-element outputs into the per-event particle list the experiment software consumes.
//   PID = argmax of the logits (L130/L156; ties -> lowest class); an element yields a candidate iff it is not a pad row and
//   its binary score is above 0.5, i.e. the binary head's logit b > 0 (the paper's rule, L156); for models without a
//   binary head (binary == NULL): iff PID != 0 (departure A23),
//   pT = pT_in exp(pT'), E = E_in exp(E')  (Eq. 2 inverted, L137-L139),  phi = atan2(sin phi, cos phi)  (L126),
//   candidates in element order, grouped per event by integer offsets (bit-exact vs the oracle).
// HBM / launch-latency bound (~90 algorithmic bytes per element): two small kernels, a stable stream
// compaction = per-block counts, then per-block prefix + scatter.  Blocks of CAND_BLOCK rows; the grid covers
// rows 0..N INCLUSIVE (row N is a virtual, never-kept row) so that every event offset, offsets[E] = N and the
// offsets of trailing empty events included, falls inside exactly one block, which writes that cand_offsets entry.
#include "cand_api.h"
#include <mutex>

namespace mlpf {

constexpr int CAND_BLOCK = 256;

// rows [row0, row0 + CAND_BLOCK) of a row-major [N, W] fp32 matrix -> shared memory, coalesced
__device__ __forceinline__ void cand_stage_rows(const float* __restrict__ g, int64_t row0, int64_t N, int W, float* s) {
    const int64_t n = (row0 + CAND_BLOCK <= N ? CAND_BLOCK : (N > row0 ? N - row0 : 0)) * (int64_t)W;
    const float* src = g + row0 * W;
    for (int64_t i = threadIdx.x; i < n; i += CAND_BLOCK) s[i] = __ldg(src + i);
}

// code[i] = PID + 1 if element i yields a candidate, else 0; block_counts[b] = candidates in block b
__global__ void __launch_bounds__(CAND_BLOCK)
k_cand_count(const float* __restrict__ X, int F, const float* __restrict__ logits, int C, const float* __restrict__ binary,
             int64_t N, uint8_t* __restrict__ code, int* __restrict__ block_counts) {
    extern __shared__ float s_lg[];                        // [CAND_BLOCK, C]
    const int64_t row0 = (int64_t)blockIdx.x * CAND_BLOCK, i = row0 + threadIdx.x;
    cand_stage_rows(logits, row0, N, C, s_lg);
    __syncthreads();
    int kept = 0;
    if (i < N) {
        const float* l = s_lg + threadIdx.x * C;           // stride C: conflict-free for odd C, 2-way at worst otherwise
        float best = l[0];
        int pid = 0;
        for (int k = 1; k < C; ++k) { const float v = l[k]; if (v > best) { best = v; pid = k; } }
        const float x0 = __ldg(X + i * F);
        const bool pad = !(x0 >= 1.0f);                     // type id clamped to 0..4 as in a0 (reading A1/A2): < 1 or NaN -> pad row
        // sigmoid(b) > 0.5  <=>  b > 0 (L156); without a binary head: class 0 = "no particle" (departure A23)
        const bool keep = !pad && (binary ? __ldg(binary + i) > 0.0f : pid != 0);
        kept = keep ? pid + 1 : 0;
        code[i] = (uint8_t)kept;
    }
    const int cnt = __syncthreads_count(kept != 0);
    if (threadIdx.x == 0) block_counts[blockIdx.x] = cnt;
}

// stable scatter of the kept rows + the cand_offsets entries of the event boundaries inside this block; the block's
// base = sum of the counts of the blocks before it (at most N / 256 L2-resident ints: cheaper than a scan launch)
__global__ void __launch_bounds__(CAND_BLOCK)
k_cand_emit(const float* __restrict__ X, int F, const float* __restrict__ regress, int64_t N,
            const int* __restrict__ offsets, int E, const uint8_t* __restrict__ code, const int* __restrict__ block_counts,
            int* __restrict__ cand_offsets, int* __restrict__ cand_elem, int* __restrict__ cand_pid,
            float4* __restrict__ cand_p4) {
    __shared__ float s_rg[CAND_BLOCK * 5];
    __shared__ int s_rank[CAND_BLOCK];                     // exclusive rank of each row inside the block
    __shared__ int s_warp[CAND_BLOCK / 32], s_base[CAND_BLOCK / 32];
    const int64_t row0 = (int64_t)blockIdx.x * CAND_BLOCK, i = row0 + threadIdx.x;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    int part = 0;
    for (int b = threadIdx.x; b < (int)blockIdx.x; b += CAND_BLOCK) part += block_counts[b];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) part += __shfl_xor_sync(0xffffffffu, part, o);
    if (lane == 0) s_base[warp] = part;
    cand_stage_rows(regress, row0, N, 5, s_rg);
    const int kept = i < N ? code[i] : 0;
    const int pid = kept - 1;
    const unsigned m = __ballot_sync(0xffffffffu, kept != 0);
    if (lane == 0) s_warp[warp] = __popc(m);
    __syncthreads();
    int before = 0, base = 0;
#pragma unroll
    for (int w = 0; w < CAND_BLOCK / 32; ++w) { before += w < warp ? s_warp[w] : 0; base += s_base[w]; }
    const int local = before + __popc(m & ((1u << lane) - 1u));
    s_rank[threadIdx.x] = local;
    if (kept != 0) {
        const float* r = s_rg + threadIdx.x * 5;
        const float pt_in = __ldg(X + i * F + 1), e_in = __ldg(X + i * F + 4);
        const int c = base + local;
        cand_elem[c] = (int)i;
        cand_pid[c] = pid;
        cand_p4[c] = make_float4(pt_in * expf(r[0]), r[1], atan2f(r[2], r[3]), e_in * expf(r[4]));
    }
    __syncthreads();
    // event boundaries with row0 <= offsets[e] < row0 + CAND_BLOCK (e = 0..E): first such e by binary search
    int lo = 0, hi = E + 1;
    while (lo < hi) { const int mid = (lo + hi) >> 1; if (offsets[mid] < row0) lo = mid + 1; else hi = mid; }
    for (int e = lo + threadIdx.x; e <= E; e += CAND_BLOCK) {
        const int64_t o = offsets[e];
        if (o >= row0 + CAND_BLOCK) break;
        cand_offsets[e] = base + s_rank[o - row0];
    }
}

int64_t cand_scratch_bytes(int64_t N, int64_t E) {
    const int64_t nb = N / CAND_BLOCK + 1;
    return ((N + 255) / 256 * 256) + ((E + 1) * 4 + 255) / 256 * 256 + (nb * 4 + 255) / 256 * 256;
}

cudaError_t launch_build_candidates(const float* X, int F, const int32_t* offsets_host, int E, const float* logits, int C,
                                    const float* regress, const float* binary, void* scratch, int32_t* cand_offsets, int32_t* cand_elem,
                                    int32_t* cand_pid, float* cand_p4, cudaStream_t st) {
    const int64_t N = offsets_host[E];
    const int nb = (int)(N / CAND_BLOCK + 1);
    uint8_t* p = (uint8_t*)scratch;
    uint8_t* code = p;                     p += (N + 255) / 256 * 256;
    int* offsets = (int*)p;                p += ((int64_t)(E + 1) * 4 + 255) / 256 * 256;
    int* block_counts = (int*)p;
    // pageable -> device async copies are staged by the runtime before returning: the caller may free offsets_host
    cudaError_t e = cudaMemcpyAsync(offsets, offsets_host, (size_t)(E + 1) * 4, cudaMemcpyHostToDevice, st);
    if (e != cudaSuccess) return e;
    k_cand_count<<<nb, CAND_BLOCK, (size_t)CAND_BLOCK * C * 4, st>>>(X, F, logits, C, binary, N, code, block_counts);
    k_cand_emit<<<nb, CAND_BLOCK, 0, st>>>(X, F, regress, N, offsets, E, code, block_counts, cand_offsets, cand_elem,
                                           cand_pid, reinterpret_cast<float4*>(cand_p4));
    return cudaGetLastError();
}

// ---- allocation-free variant (mlpf_build_candidates_static): the scratch the two kernels share lives in a file-scope
// device array, so neither the caller nor the library allocates anything (callers that cannot call cudaMalloc: tight
// serving loops, harnesses that forbid it).  Limits: N <= CAND_STATIC_MAX_N elements and E <= CAND_STATIC_MAX_E events per
// call; 283 136 bytes of device memory per GPU that loads the library, held until the process exits.  Layout = the
// caller-scratch layout at the maximum sizes: code [MAX_N] bytes | offsets [MAX_E + 1] int | block_counts [MAX_N/256 + 1] int.
// Nothing in it has to start at zero: k_cand_count writes code[0, N) and every block count the second kernel reads, the
// offsets are copied in by this call.  EVERY call shares the one array: calls that overlap on the GPU (two streams, two
// host threads without a common stream) race on it.
constexpr int64_t CAND_STATIC_MAX_N = 262144, CAND_STATIC_MAX_E = 4096;
constexpr int64_t CAND_STATIC_CODE = CAND_STATIC_MAX_N;
constexpr int64_t CAND_STATIC_OFFS = ((CAND_STATIC_MAX_E + 1) * 4 + 255) / 256 * 256;
constexpr int64_t CAND_STATIC_CNTS = ((CAND_STATIC_MAX_N / CAND_BLOCK + 1) * 4 + 255) / 256 * 256;
constexpr int64_t CAND_STATIC_BYTES = CAND_STATIC_CODE + CAND_STATIC_OFFS + CAND_STATIC_CNTS;
static __device__ __align__(256) uint8_t g_cand_scratch[CAND_STATIC_BYTES];

int64_t cand_static_max_elements() { return CAND_STATIC_MAX_N; }
int64_t cand_static_max_events() { return CAND_STATIC_MAX_E; }
int64_t cand_static_bytes() { return CAND_STATIC_BYTES; }

// The array's name is a host-side stand-in in host code: its device address comes from cudaGetSymbolAddress, asked for
// once per device with that device current (the caller's current device is the one the kernels will run on).
static cudaError_t cand_static_ptr(uint8_t** out) {
    constexpr int MAX_DEV = 64;
    static uint8_t* ptrs[MAX_DEV] = {};
    static std::mutex mu;
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= MAX_DEV) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lk(mu);
    if (!ptrs[dev]) {
        uint8_t* p = nullptr;
        e = cudaGetSymbolAddress((void**)&p, g_cand_scratch);
        if (e != cudaSuccess) return e;
        ptrs[dev] = p;
    }
    *out = ptrs[dev];
    return cudaSuccess;
}

cudaError_t launch_build_candidates_static(const float* X, int F, const int32_t* offsets_host, int E, const float* logits, int C,
                                           const float* regress, const float* binary, int32_t* cand_offsets, int32_t* cand_elem,
                                           int32_t* cand_pid, float* cand_p4, cudaStream_t st) {
    const int64_t N = offsets_host[E];
    if (N > CAND_STATIC_MAX_N || E > CAND_STATIC_MAX_E) return cudaErrorInvalidValue;      // (the entry point checks first)
    uint8_t* p = nullptr;
    cudaError_t e = cand_static_ptr(&p);
    if (e != cudaSuccess) return e;
    const int nb = (int)(N / CAND_BLOCK + 1);
    uint8_t* code = p;
    int* offsets = (int*)(p + CAND_STATIC_CODE);
    int* block_counts = (int*)(p + CAND_STATIC_CODE + CAND_STATIC_OFFS);
    e = cudaMemcpyAsync(offsets, offsets_host, (size_t)(E + 1) * 4, cudaMemcpyHostToDevice, st);
    if (e != cudaSuccess) return e;
    k_cand_count<<<nb, CAND_BLOCK, (size_t)CAND_BLOCK * C * 4, st>>>(X, F, logits, C, binary, N, code, block_counts);
    k_cand_emit<<<nb, CAND_BLOCK, 0, st>>>(X, F, regress, N, offsets, E, code, block_counts, cand_offsets, cand_elem,
                                           cand_pid, reinterpret_cast<float4*>(cand_p4));
    return cudaGetLastError();
}

}  // namespace mlpf
