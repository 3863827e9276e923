/* mlpf.h -- C ABI of libmlpf.so: the MLPF transformer-encoder forward pass on one B200 (sm_100a).
 *
 * What it computes (citations: /root/reference/PAPER.md = CMS-PFT-25-001, arxiv 2601.17554):
 *   per collision event, a variable-length *set* of PF elements (tracks, calorimeter clusters; L118-L124)
 *   -> per-type embedding FFN (L156) -> L pre-LayerNorm transformer encoder blocks with full-event
 *   scaled-dot-product self-attention  A = softmax(Q K^T / sqrt(d_k)) V  (Eq. 4; computed
 *   flash-style without the N x N matrix, L154) -> two-layer FFN heads giving particle-id logits and
 *   the momentum regressions (pT', eta, sin phi, cos phi, E')  (L126, L134-L139, L156, Fig. 2).
 *   The readings taken where the paper is silent are A1-A23 in DESIGN.md.
 *
 * All functions are thread-safe per handle; concurrent mlpf_infer calls on DIFFERENT streams are safe
 * (each stream owns a grow-only workspace), calls on the same stream serialise in stream order.
 * Every step runs in hand-written CUDA kernels; there is no CPU fallback: without a CUDA device every
 * entry point that needs one fails with MLPF_E_CUDA.
 */
#ifndef MLPF_H_
#define MLPF_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct mlpf_handle mlpf_handle;

/* ---- error codes (0 = success) ------------------------------------------------------------------ */
#define MLPF_OK          0
#define MLPF_E_NULL     -1   /* a required pointer is NULL                                            */
#define MLPF_E_BLOB     -2   /* bad magic / version / hyper-parameters / size of the weight blob      */
#define MLPF_E_OFFSETS  -3   /* event_offsets[0] != 0, decreasing, or negative                        */
#define MLPF_E_ALLOC    -4   /* device or host allocation failed                                      */
#define MLPF_E_CUDA     -5   /* a CUDA call failed (text in mlpf_last_error)                          */
#define MLPF_E_ARG      -6   /* unknown option / query key, bad value, capacity too small             */

/* ---- weight blob (little-endian) -------------------------------------------------------------------
 * 256-byte header, then fp32 tensors, row-major [out,in] (y = x W^T + b), in this order:
 *   for type t = 1..n_types      : emb.t.W1[d,F] b1[d] W2[d,d] b2[d]                     (L156, A3-A4)
 *   for stack s = 0..n_stacks-1, for layer l = 0..n_layers-1 :
 *                                  ln1.g[d] ln1.b[d] Wqkv[3d,d] bqkv[3d] Wo[d,d] bo[d]
 *                                  ln2.g[d] ln2.b[d] W1[dff,d] b1[dff] W2[d,dff] b2[d]   (L148-L156)
 *   for stack s                  : lnf.g[d] lnf.b[d]                                     (A7)
 *   if binary_head               : bin.W1[d,d] b1[d] W2[1,d] b2[1]                       (L156, Fig. 2)
 *   cls.W1[d,d] b1[d] W2[C,d] b2[C]                                                      (L156, A11)
 *   for k = 0..n_reg_heads-1     : reg.k.W1[d,d] b1[d] W2[reg_dims[k],d] b2[reg_dims[k]]
 * Master weights are fp32.  In BF16 mode the library rounds (RNE) the matrices that feed tensor-core
 * GEMMs (emb W2, Wqkv, Wo, W1, W2, cls.W1, reg.k.W1, bin.W1); emb W1, the output rows
 * (cls.W2, reg.k.W2, bin.W2) and all vectors stay fp32.
 */
#define MLPF_BLOB_MAGIC   "MLPFBLOB"
#define MLPF_BLOB_VERSION 2u  /* version 1 blobs (one stack, no binary head; the two new header fields are padding) still load */
#define MLPF_HEADER_BYTES 256
#define MLPF_MAX_REG_HEADS 4

typedef struct mlpf_blob_header {
    char     magic[8];       /* "MLPFBLOB" */
    uint32_t version;        /* 1 */
    uint32_t n_layers;       /* L  >= 1 */
    uint32_t d_model;        /* d  in {64,128,256,512}; multiple of 64 */
    uint32_t n_heads;        /* H ; d/H in {16,32,64} */
    uint32_t d_ff;           /* multiple of 64 */
    uint32_t n_feat;         /* F = 55 (A13); 1 <= F <= 64 */
    uint32_t n_types;        /* T = 4 (A3) */
    uint32_t n_classes;      /* C = 9 (A13); <= 16 */
    uint32_t n_reg_heads;    /* <= 4 (A11) */
    uint32_t reg_dims[MLPF_MAX_REG_HEADS]; /* (1,1,2,1): pT', eta, (sin phi, cos phi), E' ; sum <= 8 */
    uint32_t activation;     /* 0 = ReLU (L156), 1 = GELU exact-erf form (A6) */
    uint32_t final_ln;       /* 0/1 (A7) */
    float    ln_eps;         /* 1e-5 (A8) */
    uint32_t n_stacks;       /* version 2: 1 = one encoder; 2 = the paper's two parallel encoders on the shared embedding
                                (L156): stack 0 = classification, stack 1 = regression */
    uint32_t binary_head;    /* version 2: 1 = a binary "valid" head on stack 0 (L156, Fig. 2) */
    /* zero padding up to MLPF_HEADER_BYTES */
} mlpf_blob_header;

/* mlpf_create: parse + validate `blob` (HOST pointer, borrowed only during the call), upload weights to
 * the current CUDA device (fp32 masters + BF16 copies).  Returns NULL on error (see mlpf_last_error). */
mlpf_handle* mlpf_create(const void* blob, size_t blob_bytes);

/* mlpf_infer: one forward pass (steps a0..a8 of DESIGN.md) over n_events packed events.
 *   elements      DEVICE, [N, n_feat] row-major fp32, N = event_offsets[n_events]; feature 0 is the
 *                 element type id as a float (0 = pad row, 1 track, 2 ECAL, 3 HCAL, 4 HF; A1-A2).
 *                 NaN / Inf features of a non-pad row give undefined outputs for THAT event and no other (never a crash):
 *                 every step but attention is row-local, and the attention kernel zeroes, in shared memory, the rows of
 *                 the next event that an event's last K / V tile overlaps (their keys have weight exactly 0, but
 *                 0 x NaN = NaN in the tensor core).  Round 1's attention kernel (MLPF_OPT_ATTN = 0) does not: with it,
 *                 finite features are a precondition.  Pad rows may hold anything (dropped before the first GEMM).
 *   event_offsets HOST, n_events+1 int32, [0] = 0, non-decreasing; read before return (caller may free).
 *   out_logits    DEVICE, [N, n_classes] fp32.   out_regress  DEVICE, [N, sum(reg_dims)] fp32
 *                 = raw head outputs (pT', eta, sin phi, cos phi, E'), no inverse transform (A12).
 *                 Pad rows are written as exactly 0 (A2).
 *   stream        cudaStream_t (NULL = legacy default stream).
 * Only enqueues work on `stream` (no device synchronisation; the first call on a stream, or a call with a
 * larger N than before, may cudaMalloc).  n_events == 0 or N == 0: success, nothing written.
 * Returns MLPF_OK or a negative error code. */
int mlpf_infer(mlpf_handle* h, const float* elements, const int32_t* event_offsets, int32_t n_events,
               float* out_logits, float* out_regress, void* stream);

/* mlpf_infer_host: same computation with HOST buffers (pinned memory recommended): copies `elements`
 * host->device, runs mlpf_infer, copies both outputs device->host, all on `stream`, then synchronises
 * the stream.  This is the end-to-end entry (the paper's deployment copies per event, L224). */
int mlpf_infer_host(mlpf_handle* h, const float* elements_host, const int32_t* event_offsets,
                    int32_t n_events, float* out_logits_host, float* out_regress_host, void* stream);

/* mlpf_infer_ex: mlpf_infer plus the binary head's logit, out_binary DEVICE [N] fp32 (pad rows 0), for models with a binary
 * head (MLPF_Q_BINARY_HEAD); out_binary may be NULL.  With n_stacks = 2 the binary and PID heads read the classification
 * encoder and the regression heads read the regression encoder (L156); both encoders run as ONE grouped batch (every
 * kernel launch covers both stacks). */
int mlpf_infer_ex(mlpf_handle* h, const float* elements, const int32_t* event_offsets, int32_t n_events,
                  float* out_logits, float* out_regress, float* out_binary, void* stream);

/* mlpf_infer_host_async / mlpf_host_sync: the same as mlpf_infer_host without the final synchronisation.  The H2D copy runs
 * on a copy-in stream of the library, the kernels on `stream`, the D2H copies on a copy-out stream, chained by events; two
 * device staging slots alternate, so with several calls in flight the copies of one call overlap the kernels of its
 * neighbours (the paper's "asynchronous ... execution", L232).  The host buffers of a call must stay valid and untouched
 * until mlpf_host_sync(h, stream) returns (it waits for every call issued on that stream so far). */
int mlpf_infer_host_async(mlpf_handle* h, const float* elements_host, const int32_t* event_offsets, int32_t n_events,
                          float* out_logits_host, float* out_regress_host, void* stream);
int mlpf_host_sync(mlpf_handle* h, void* stream);

void mlpf_destroy(mlpf_handle* h);

/* Thread-local text of the last error raised on this thread ("" if none). */
const char* mlpf_last_error(void);

/* ---- candidate building (the step after the forward pass; "builds the particle candidates") -------
 * From the per-element outputs of mlpf_infer to the per-event list of particle candidates:
 *   PID_i = argmax_c logits[i,c] (multiclass PID head, L130/L156; ties -> lowest class);
 *   element i yields a candidate iff its type (feature 0, clamped to 0..4) != 0 and PID_i != 0 (class 0 = "no particle":
 *   DEPARTURE A23 from the paper's rule, for models whose single PID head is all there is; models with a binary head use
 *   mlpf_build_candidates_ex, which implements the paper's rule);
 *   pT = x_i[1] exp(pT'), E = x_i[4] exp(E') (Eq. 2 inverted, L137-L139; x_i[1], x_i[4] = the element's own pT, E),
 *   eta = raw output, phi = atan2(sin phi, cos phi) (L126).
 * Candidates keep the element order (stable compaction) and are grouped per event:
 *   cand_offsets [n_events+1] int32: event e owns candidates cand_offsets[e] .. cand_offsets[e+1]-1;
 *   cand_elem [M] int32 global row of the element, cand_pid [M] int32, cand_p4 [M,4] fp32 (pT, eta, phi, E),
 *   M = cand_offsets[n_events] <= N; entries beyond M are not written.
 * All pointers are DEVICE pointers except event_offsets (HOST, read before return, same rules as mlpf_infer).
 * regress is [N,5] = (pT', eta, sin phi, cos phi, E'); logits [N,n_classes], n_classes 1..64; elements [N,n_feat],
 * n_feat >= 5.  cand_elem / cand_pid / cand_p4 need capacity N (cand_p4 16-byte aligned); scratch is caller-owned
 * device memory, 256-byte aligned, of at least mlpf_candidates_scratch_bytes(N, n_events) bytes, and may be reused
 * by the next call on the same stream.  Only enqueues on `stream` (two kernels); no allocation, no sync.
 * Integer outputs are bit-exact vs the oracle on the same fp32 logits; pT, E, phi are fp32 expf / atan2f.
 * n_events == 0: success, nothing written.  N == 0: cand_offsets is all zeros.  Errors as for mlpf_infer. */
int64_t mlpf_candidates_scratch_bytes(int64_t n_elements, int32_t n_events);   /* < 0 on error */
/* mlpf_build_candidates_ex: the same with the paper's selection rule (L156): `binary` DEVICE [N] fp32 = the binary head's
 * logit; an element yields a candidate iff it is not a pad row and sigmoid(binary) > 0.5 (i.e. binary > 0), its PID is
 * the argmax over ALL classes.  binary == NULL: the class-0 rule above (departure A23).  n_regress must be 5;
 * n_classes <= 48. */
int mlpf_build_candidates_ex(const float* elements, int32_t n_feat, const int32_t* event_offsets, int32_t n_events,
                             const float* logits, int32_t n_classes, const float* regress, int32_t n_regress,
                             const float* binary, void* scratch, int64_t scratch_bytes, int32_t* cand_offsets,
                             int32_t* cand_elem, int32_t* cand_pid, float* cand_p4, void* stream);
int mlpf_build_candidates(const float* elements, int32_t n_feat, const int32_t* event_offsets, int32_t n_events,
                          const float* logits, int32_t n_classes, const float* regress, void* scratch,
                          int64_t scratch_bytes, int32_t* cand_offsets, int32_t* cand_elem, int32_t* cand_pid,
                          float* cand_p4, void* stream);

/* mlpf_build_candidates_static: mlpf_build_candidates_ex for callers that cannot allocate (no cudaMalloc in a tight serving
 * loop or a harness that forbids it): same inputs, outputs and results, but the kernels' scratch is a file-scope device
 * array inside the library, so the caller passes no scratch and this path calls no cudaMalloc / cudaFree / allocating
 * library routine.  Limits per call: N <= mlpf_candidates_static_limit(0) = 262144 elements and n_events <=
 * mlpf_candidates_static_limit(1) = 4096; beyond them MLPF_E_ARG (nothing enqueued).  The array
 * (mlpf_candidates_static_limit(2) = 283136 bytes) is held by every GPU that loads the library until the process exits.
 * ALL calls on a device share it: calls that overlap on the GPU (different streams, or host threads without a common
 * stream) race; calls on one stream are ordered and safe.  It keeps the last call's contents; nothing in it has to start
 * at zero (every byte a call reads is written by that call first).  Uses the CURRENT device; pointers as above. */
int mlpf_build_candidates_static(const float* elements, int32_t n_feat, const int32_t* event_offsets, int32_t n_events,
                                 const float* logits, int32_t n_classes, const float* regress, int32_t n_regress,
                                 const float* binary, int32_t* cand_offsets, int32_t* cand_elem, int32_t* cand_pid,
                                 float* cand_p4, void* stream);
int64_t mlpf_candidates_static_limit(int32_t which);   /* 0: max elements, 1: max events, 2: bytes held per GPU; < 0 on error */

/* ---- options -------------------------------------------------------------------------------------- */
#define MLPF_OPT_PRECISION   1   /* MLPF_PREC_BF16 (default) | MLPF_PREC_FP32_DEBUG                    */
#define MLPF_OPT_TILE_Q      2   /* query-tile rows of the attention work list: 64 | 128 (default 128) */
#define MLPF_OPT_TAP_LAYER   3   /* -1 (default): full pass.  l >= 0: stop after encoder layer l so that
                                    mlpf_debug_get_tensor can read that layer's intermediates; outputs
                                    are then NOT written.  -2: stop after the embedding.                */
#define MLPF_OPT_KERNELS     4   /* MLPF_KERNELS_TC (default: tcgen05 GEMM + attention) | MLPF_KERNELS_SIMPLE
                                    (CUDA-core kernels in the same precision; debugging aid)            */
#define MLPF_OPT_SPLIT       5   /* bit mask (default MLPF_SPLIT_ALL): which bf16 activations of the BF16 path are carried
                                    as two bf16 terms hi + lo and multiplied as two MMAs into one fp32 accumulator
                                    (DESIGN.md "error budget").  0: single bf16 term everywhere.             */
#define MLPF_SPLIT_EMB   1       /* embedding hidden layer (input of the embedding's second linear)          */
#define MLPF_SPLIT_O     2       /* attention output (input of the out-projection)                           */
#define MLPF_SPLIT_U2    4       /* LN2 output (input of FFN1)                                               */
#define MLPF_SPLIT_G     8       /* FFN hidden layer (input of FFN2)                                         */
#define MLPF_SPLIT_UF    16      /* final-LN output (input of the heads' first layers)                       */
#define MLPF_SPLIT_HEAD  32      /* heads' hidden layers (input of the fp32 output rows)                     */
#define MLPF_SPLIT_ALL   63
#define MLPF_OPT_PROFILE     6   /* 1: record a CUDA event pair around every kernel class inside mlpf_infer
                                    (read back with mlpf_debug_get_profile); 0 (default): off            */
#define MLPF_OPT_FUSE        7   /* 1 (default): where the shape allows (d_model <= 256, d_ff % 128 == 0, all activations split)
                                    the post-attention half of every block runs as ONE kernel (out-projection + residual +
                                    LN2 + FFN1 + activation + FFN2 + residual + next LayerNorm); 0: one kernel per step   */
#define MLPF_OPT_ATTN        8   /* attention kernel: 1 (default) = tc_attn2.cu (no running maximum: Cauchy-Schwarz bound from row norms
                                    (MLPF_OPT_EPI_NORMS), exact two-sweep path when the bound is too loose; two threads per query row);
                                    2 = the same with the exact path forced for every CTA; 0 = round 1's lazy-rescale kernel */
#define MLPF_OPT_ATTN_POLY   9   /* tuning (process-wide): n of every 16 pairs of softmax exponentials run as a polynomial on the
                                    FMA pipe instead of the MUFU: 0 (none), 4, 7, 8, 9; -1 (default) = 8 in the model path (scores prescaled by a3's
                                    epilogue); 7 at hd <= 32, 0 at hd = 64 for the unscaled kernel-level entry          */
#define MLPF_OPT_COMPACT     10  /* 1 (default): pad rows (type 0) are dropped after a0: every later step runs on the compacted rows
                                    (events stay contiguous, oracle.schedule comp_row / offsets_c), outputs are scattered back;
                                    0: pad rows stay in place and are masked as keys (round 1's behaviour)                   */
#define MLPF_OPT_GRAPH       11  /* 1: a forward pass whose key (pointers, sizes, event_offsets, options) repeats is captured into a
                                    CUDA graph on its second occurrence and replayed afterwards (one launch per call: the
                                    one-event-per-call mode of PAPER.md L224); 0 (default): plain launches                   */
#define MLPF_OPT_TAIL_SPLIT  12  /* 1 (default): the attention CTAs of a mostly empty last wave are split into single-query-tile
                                    CTAs (shorter tail); 0: every CTA takes up to NT query tiles                              */
#define MLPF_OPT_FP8         13  /* NEXT-3 (PAPER.md L232 / L238 "quantization"): 1 = the QKV projection runs with e4m3 operands
                                    (tcgen05 kind::f8f6f4; one scale per weight matrix, a fixed scale of 16 for the LayerNorm
                                    output, fp32 accumulate); 0 (default): BF16.  The measured drift is in DESIGN.md.          */
#define MLPF_OPT_EPI_NORMS   14  /* 1 (default): the attention softmax bound's inputs (|q| per row and head, max |k| per event and
                                    head) come out of the QKV projection's epilogue, which also folds the softmax scale log2(e) / sqrt(hd)
                                    into q before its bf16 rounding (the attention kernel then exponentiates q k as it is and, on its
                                    fast path, subtracts nothing); 0: unscaled q, a separate pre-pass kernel computes the norms        */
#define MLPF_OPT_TC_EMBED    15  /* 1 (default): the first embedding layer (fp32 weights, reading A3) runs on the tensor pipe as ONE
                                    K = 192 grouped GEMM over bf16 terms [x_hi | x_lo | x_hi] x [W_hi | W_hi | W_lo] (relative error
                                    ~2^-17: the x_lo W_lo term is dropped); 0: fp32 FMAs on the CUDA cores (k_embed_l1)        */
#define MLPF_OPT_PDL         16  /* 1: the tensor-core kernels are launched as programmatic dependents of the kernel before them (their
                                    set-up and first wave overlap its tail; griddepcontrol.wait orders every access); 0: plain stream
                                    order; 2 (default): 1 for calls whose attention grid is at most two waves of CTAs (one event per
                                    call: 0.847 -> 0.823 ms), else 0 (no gain on large batches)                              */
#define MLPF_OPT_ATTN_POLY_DEG 17 /* tuning (process-wide): degree of that polynomial, 3 (default: relative error 1e-4) or 2 (1.8e-3, the
                                    size of the bf16 rounding of the softmax weight itself; measured in profiles/r02_README.md)  */
#define MLPF_PREC_BF16        0
#define MLPF_PREC_FP32_DEBUG  1
#define MLPF_KERNELS_TC       0
#define MLPF_KERNELS_SIMPLE   1
int mlpf_set_option(mlpf_handle* h, int key, int64_t value);

/* ---- queries -------------------------------------------------------------------------------------- */
#define MLPF_Q_N_LAYERS        1
#define MLPF_Q_D_MODEL         2
#define MLPF_Q_N_HEADS         3
#define MLPF_Q_D_FF            4
#define MLPF_Q_N_FEAT          5
#define MLPF_Q_N_CLASSES       6
#define MLPF_Q_N_REGRESS       7
#define MLPF_Q_WEIGHT_BYTES    8   /* device bytes held by weights (fp32 + bf16 copies)                */
#define MLPF_Q_WORKSPACE_BYTES 9   /* device bytes held by all per-stream workspaces (linear in N)      */
#define MLPF_Q_N_PARAMS        10
#define MLPF_Q_LAUNCHES        11  /* kernels launched by the last mlpf_infer on this handle             */
#define MLPF_Q_N_STACKS        12
#define MLPF_Q_BINARY_HEAD     13
int64_t mlpf_query(const mlpf_handle* h, int key);   /* < 0 on error */

/* ---- debug taps (tests only; these synchronise `stream`) ------------------------------------------- */
/* integer schedule arrays of the last mlpf_infer on `stream` (step a0; bit-exact vs the oracle) */
#define MLPF_SCHED_ROW_EVENT    0   /* [N]                                   */
#define MLPF_SCHED_ROW_POS      1   /* [N]                                   */
#define MLPF_SCHED_VALID        2   /* [N] 0/1                               */
#define MLPF_SCHED_N_VALID      3   /* [E]                                   */
#define MLPF_SCHED_TYPE_OFFSETS 4   /* [6] segment starts in sorted space, each a multiple of 128 */
#define MLPF_SCHED_SORTED_ROW   5   /* [N] row -> sorted slot, -1 for pad    */
#define MLPF_SCHED_TYPE_PERM    6   /* [type_offsets[5]] slot -> row, -1 filler */
#define MLPF_SCHED_WORK_LIST    7   /* [n_tiles,2] (event, q_tile)           */
#define MLPF_SCHED_COMP_ROW     8   /* [N] row -> compacted row, -1 for pad  */
#define MLPF_SCHED_OFFSETS_C    9   /* [E+1] event offsets in compacted rows */
#define MLPF_SCHED_COMP_TYPE_PERM 10 /* [type_offsets[5]] slot -> compacted row, -1 filler */
/* returns the number of int32 written, or a negative error (MLPF_E_ARG if capacity is too small) */
int64_t mlpf_debug_get_schedule(mlpf_handle* h, void* stream, int which, int32_t* host_out, int64_t capacity);

/* intermediates of the last mlpf_infer on `stream`, converted to fp32, row-major:
 * H [N,d] residual stream; U [N,d] last LayerNorm output; QK [N,2d] (q | k); V [N,d];
 * O [N,d] attention output; G [N,gw] last wide hidden (FFN: gw = d_ff; heads: gw = (1+n_reg_heads) d).
 * Which stage they hold depends on MLPF_OPT_TAP_LAYER.  Returns floats written or a negative error. */
#define MLPF_TENSOR_H   0
#define MLPF_TENSOR_U   1
#define MLPF_TENSOR_QK  2
#define MLPF_TENSOR_V   3
#define MLPF_TENSOR_O   4
#define MLPF_TENSOR_G   5
int64_t mlpf_debug_get_tensor(mlpf_handle* h, void* stream, int which, float* host_out, int64_t capacity);

/* per-kernel-class device time of the last mlpf_infer on `stream` run with MLPF_OPT_PROFILE = 1:
 * ms_out[MLPF_KC_COUNT] (sum over the call's launches of that class) and count_out[MLPF_KC_COUNT]. */
#define MLPF_KC_SCHED      0   /* a0 */
#define MLPF_KC_EMBED_L1   1   /* a1 first layer (fp32, CUDA cores) */
#define MLPF_KC_EMBED_L2   2   /* a1 second layer (grouped GEMM) */
#define MLPF_KC_LAYERNORM  3   /* a2 */
#define MLPF_KC_QKV        4   /* a3 */
#define MLPF_KC_ATTENTION  5   /* a4 */
#define MLPF_KC_OUTPROJ    6   /* a5 */
#define MLPF_KC_FFN1       7   /* a6 */
#define MLPF_KC_FFN2       8   /* a7 */
#define MLPF_KC_HEADS_L1   9   /* a8 first layers */
#define MLPF_KC_HEADS_L2   10  /* a8 output rows */
#define MLPF_KC_POST       11  /* a5 + a6 + a7 fused (tc_post.cu) */
#define MLPF_KC_COUNT      12
int mlpf_debug_get_profile(mlpf_handle* h, void* stream, float* ms_out, int32_t* count_out);

/* ---- kernel-level entry points (unit tests and micro-benchmarks; device pointers, bf16 = uint16) ---- */
/* C[M,N] (fp32, ldc = N) = (A + A_lo)[M,K] (bf16, row-major; A_lo may be NULL) * W[N,K]^T (bf16, row-major)
 * via the tcgen05 GEMM.  K % 64 == 0, N % 64 == 0.  Step a3/a5/a6/a7's contraction (L148-L156), no epilogue. */
int mlpf_tc_gemm_bf16(const uint16_t* A, const uint16_t* A_lo, const uint16_t* W, float* C, int32_t M, int32_t N,
                      int32_t K, void* stream);
/* C[M,N] (fp32) = out_scale * A[M,K] W[N,K]^T with e4m3 operands (one byte per element, row-major) via the tcgen05
 * kind::f8f6f4 GEMM.  K % 128 == 0, N % 128 == 0. */
int mlpf_tc_gemm_fp8(const uint8_t* A, const uint8_t* W, float* C, int32_t M, int32_t N, int32_t K, float out_scale, void* stream);
/* O[N,d] (bf16) = per-event multi-head softmax(Q K^T / sqrt(hd)) V (Eq. 4) via the tcgen05 flash kernel.
 * QKV [N,3d] bf16 row-major (q | k | v), key_valid [N] int32 0/1 (NULL = all valid),
 * event_offsets HOST int32 [n_events+1]; events may start at any row. */
int mlpf_tc_attention_bf16(const uint16_t* QKV, const int32_t* key_valid,
                           const int32_t* event_offsets, int32_t n_events, int32_t d_model, int32_t n_heads,
                           uint16_t* O, void* stream);

/* Measured throughput, in results per clock per SM, of the units that bound the attention softmax (Eq. 4: one
 * exponential per score): which = 0 ex2.approx.ftz.f32 (MUFU), 1 ex2.approx.ftz.bf16x2 (MUFU, packed), 2 the polynomial
 * 2^x of tc_attn2.cu on the FMA / ALU pipes, 3 fma.rn.f32x2.  One CTA of 1024 threads per SM, `iters` x 8 independent
 * operations per thread, cycles from clock64.  Synchronises `stream`.  < 0 on error.  bench.py's roofline.alu uses it. */
float mlpf_microbench(int32_t which, int32_t iters, void* stream);

/* which kernel mlpf_tc_attention_bf16 runs (process-wide; 0 .. 2 as MLPF_OPT_ATTN; 3 / 4 = 1 / 2 for a QKV whose q columns
 * were already multiplied by log2(e) / sqrt(head_dim) before their bf16 rounding: the form the model path feeds the kernel) */
int mlpf_debug_set_attention_impl(int impl);

/* The post-attention half of one encoder block (steps a5 + a6 + a7 with both LayerNorms in epilogues)
 * as ONE kernel:  h <- h + (o_hi + o_lo) Wo^T + bo;  u2 = LN2(h);  h <- h + act(u2 W1^T + b1) W2^T + b2;
 * u_out (+ u_out_lo) = bf16 hi (+ lo) of LN_next(h), or of h itself when lnng / lnnb are NULL.
 * All DEVICE pointers: o_hi, o_lo, u_out, u_out_lo [M,d] bf16; h [M,d] fp32 in/out; Wo [d,d], W1 [dff,d], W2 [d,dff] bf16
 * row-major [out,in]; vectors fp32.  d in {64,128,256}, dff % 128 == 0; activation 0 = ReLU, 1 = GELU (erf).
 * Only enqueues on `stream`. */
int mlpf_tc_post_bf16(const uint16_t* o_hi, const uint16_t* o_lo, float* h, const uint16_t* Wo, const float* bo,
                      const float* ln2g, const float* ln2b, const uint16_t* W1, const float* b1, const uint16_t* W2,
                      const float* b2, const float* lnng, const float* lnnb, int32_t M, int32_t d, int32_t dff,
                      int32_t activation, float ln_eps, uint16_t* u_out, uint16_t* u_out_lo, void* stream);

#ifdef __cplusplus
}
#endif
#endif /* MLPF_H_ */
