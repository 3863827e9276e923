"""paper_2601_17554_b200 -- thin ctypes binding over libmlpf.so (include/mlpf.h).

Argument marshalling only: every step of the MLPF encoder forward pass runs in
the library's CUDA kernels.  torch is used for device memory and streams.  There is no CPU fallback:
importing works without a GPU (so that the symbols can be checked), creating a model does not.
"""
from __future__ import annotations
import ctypes as C
import os
import numpy as np

from .blob import pack_blob

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libmlpf.so")

# include/mlpf.h constants
OK = 0
OPT_PRECISION, OPT_TILE_Q, OPT_TAP_LAYER, OPT_KERNELS, OPT_SPLIT, OPT_PROFILE, OPT_FUSE, OPT_ATTN, OPT_ATTN_POLY, OPT_COMPACT, OPT_GRAPH, OPT_TAIL_SPLIT, OPT_FP8, OPT_EPI_NORMS, OPT_TC_EMBED, OPT_PDL, OPT_ATTN_POLY_DEG = 1, 2, 3, 4, 5, 6, 7, 8, 9, 10, 11, 12, 13, 14, 15, 16, 17
PREC_BF16, PREC_FP32_DEBUG = 0, 1
KERNELS_TC, KERNELS_SIMPLE = 0, 1
Q_N_LAYERS, Q_D_MODEL, Q_N_HEADS, Q_D_FF, Q_N_FEAT, Q_N_CLASSES, Q_N_REGRESS = 1, 2, 3, 4, 5, 6, 7
Q_WEIGHT_BYTES, Q_WORKSPACE_BYTES, Q_N_PARAMS, Q_LAUNCHES, Q_N_STACKS, Q_BINARY_HEAD = 8, 9, 10, 11, 12, 13
SCHED = dict(row_event=0, row_pos=1, valid=2, n_valid=3, type_offsets=4, sorted_row=5, type_perm=6, work_list=7,
             comp_row=8, offsets_c=9, comp_type_perm=10)
TENSOR = dict(H=0, U=1, QK=2, V=3, O=4, G=5)
KERNEL_CLASSES = ["sched", "embed_l1", "embed_l2", "layernorm", "qkv", "attention", "outproj", "ffn1", "ffn2",
                  "heads_l1", "heads_l2", "post"]

EXPORTS = ["mlpf_create", "mlpf_infer", "mlpf_infer_ex", "mlpf_build_candidates_ex", "mlpf_infer_host", "mlpf_infer_host_async",
           "mlpf_host_sync", "mlpf_destroy", "mlpf_last_error", "mlpf_set_option",
           "mlpf_query", "mlpf_debug_get_schedule", "mlpf_debug_get_tensor", "mlpf_debug_get_profile", "mlpf_tc_gemm_bf16",
           "mlpf_tc_attention_bf16", "mlpf_debug_set_attention_impl", "mlpf_microbench", "mlpf_tc_gemm_fp8", "mlpf_tc_post_bf16", "mlpf_candidates_scratch_bytes", "mlpf_build_candidates",
           "mlpf_build_candidates_static", "mlpf_candidates_static_limit"]

_lib = None


def lib():
    """Load libmlpf.so (built in-tree by paper_2601_17554_b200.build); fails loudly if it is missing."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise RuntimeError(f"{LIB_PATH} is missing: run `python -m paper_2601_17554_b200.build` "
                           "(there is no CPU fallback)")
    L = C.CDLL(LIB_PATH)
    vp, i32, i64 = C.c_void_p, C.c_int32, C.c_int64
    L.mlpf_create.restype = vp
    L.mlpf_create.argtypes = [vp, C.c_size_t]
    L.mlpf_infer.restype = C.c_int
    L.mlpf_infer.argtypes = [vp, vp, vp, i32, vp, vp, vp]
    L.mlpf_infer_ex.restype = C.c_int
    L.mlpf_infer_ex.argtypes = [vp, vp, vp, i32, vp, vp, vp, vp]
    L.mlpf_build_candidates_ex.restype = C.c_int
    L.mlpf_build_candidates_ex.argtypes = [vp, i32, vp, i32, vp, i32, vp, i32, vp, vp, i64, vp, vp, vp, vp, vp]
    L.mlpf_infer_host.restype = C.c_int
    L.mlpf_infer_host.argtypes = [vp, vp, vp, i32, vp, vp, vp]
    L.mlpf_infer_host_async.restype = C.c_int
    L.mlpf_infer_host_async.argtypes = [vp, vp, vp, i32, vp, vp, vp]
    L.mlpf_host_sync.restype = C.c_int
    L.mlpf_host_sync.argtypes = [vp, vp]
    L.mlpf_destroy.restype = None
    L.mlpf_destroy.argtypes = [vp]
    L.mlpf_last_error.restype = C.c_char_p
    L.mlpf_last_error.argtypes = []
    L.mlpf_set_option.restype = C.c_int
    L.mlpf_set_option.argtypes = [vp, C.c_int, i64]
    L.mlpf_query.restype = i64
    L.mlpf_query.argtypes = [vp, C.c_int]
    L.mlpf_debug_get_schedule.restype = i64
    L.mlpf_debug_get_schedule.argtypes = [vp, vp, C.c_int, vp, i64]
    L.mlpf_debug_get_tensor.restype = i64
    L.mlpf_debug_get_tensor.argtypes = [vp, vp, C.c_int, vp, i64]
    L.mlpf_debug_get_profile.restype = C.c_int
    L.mlpf_debug_get_profile.argtypes = [vp, vp, vp, vp]
    L.mlpf_tc_gemm_bf16.restype = C.c_int
    L.mlpf_tc_gemm_bf16.argtypes = [vp, vp, vp, vp, i32, i32, i32, vp]
    L.mlpf_tc_attention_bf16.restype = C.c_int
    L.mlpf_tc_attention_bf16.argtypes = [vp, vp, vp, i32, i32, i32, vp, vp]
    L.mlpf_tc_gemm_fp8.restype = C.c_int
    L.mlpf_tc_gemm_fp8.argtypes = [vp, vp, vp, i32, i32, i32, C.c_float, vp]
    L.mlpf_microbench.restype = C.c_float
    L.mlpf_microbench.argtypes = [i32, i32, vp]
    L.mlpf_debug_set_attention_impl.restype = C.c_int
    L.mlpf_debug_set_attention_impl.argtypes = [C.c_int]
    L.mlpf_tc_post_bf16.restype = C.c_int
    L.mlpf_tc_post_bf16.argtypes = [vp] * 13 + [i32, i32, i32, i32, C.c_float, vp, vp, vp]
    L.mlpf_candidates_scratch_bytes.restype = i64
    L.mlpf_candidates_scratch_bytes.argtypes = [i64, i32]
    L.mlpf_build_candidates_static.restype = C.c_int
    L.mlpf_build_candidates_static.argtypes = [vp, i32, vp, i32, vp, i32, vp, i32, vp, vp, vp, vp, vp, vp]
    L.mlpf_candidates_static_limit.restype = i64
    L.mlpf_candidates_static_limit.argtypes = [i32]
    L.mlpf_build_candidates.restype = C.c_int
    L.mlpf_build_candidates.argtypes = [vp, i32, vp, i32, vp, i32, vp, vp, i64, vp, vp, vp, vp, vp]
    _lib = L
    return L


class MlpfError(RuntimeError):
    pass


def _check(rc):
    if rc < 0:
        raise MlpfError(f"libmlpf error {rc}: {lib().mlpf_last_error().decode()}")
    return rc


def _stream_ptr(stream):
    if stream is None:
        import torch
        stream = torch.cuda.current_stream()
    return C.c_void_p(stream.cuda_stream)


class Mlpf:
    """One model instance (mlpf_create ... mlpf_destroy)."""

    def __init__(self, W: dict, m):
        self._h = None
        blob = pack_blob(W, m)
        self.m = m
        buf = C.create_string_buffer(blob, len(blob))
        h = lib().mlpf_create(C.cast(buf, C.c_void_p), len(blob))
        if not h:
            raise MlpfError("mlpf_create failed: " + lib().mlpf_last_error().decode())
        self._h = C.c_void_p(h)
        self.n_classes = int(self.query(Q_N_CLASSES))
        self.n_regress = int(self.query(Q_N_REGRESS))
        self.n_feat = int(self.query(Q_N_FEAT))
        self.d_model = int(self.query(Q_D_MODEL))
        self.binary_head = bool(self.query(Q_BINARY_HEAD))

    def close(self):
        if self._h is not None:
            lib().mlpf_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_option(self, key, value):
        _check(lib().mlpf_set_option(self._h, key, int(value)))

    def query(self, key):
        return _check(lib().mlpf_query(self._h, key))

    def infer(self, elements, event_offsets, out_logits=None, out_regress=None, stream=None, out_binary=None, with_binary=False):
        """elements: CUDA float32 tensor [N, n_feat]; event_offsets: host int32 array [E+1].
        Returns (logits [N,C], regress [N,R]) CUDA float32 tensors (enqueued on `stream`); with with_binary=True (models with
        a binary head) also the binary head's logit [N]."""
        import torch
        assert elements.is_cuda and elements.dtype == torch.float32 and elements.is_contiguous()
        off = np.ascontiguousarray(event_offsets, dtype=np.int32)
        N = elements.shape[0]
        assert len(off) >= 1 and int(off[-1]) == N, "event_offsets[-1] must equal the number of element rows"
        if with_binary or out_binary is not None:
            if out_logits is None:
                out_logits = torch.empty((N, self.n_classes), dtype=torch.float32, device=elements.device)
            if out_regress is None:
                out_regress = torch.empty((N, self.n_regress), dtype=torch.float32, device=elements.device)
            if out_binary is None:
                out_binary = torch.empty((N,), dtype=torch.float32, device=elements.device)
            _check(lib().mlpf_infer_ex(self._h, C.c_void_p(elements.data_ptr()), off.ctypes.data_as(C.c_void_p), len(off) - 1,
                                       C.c_void_p(out_logits.data_ptr()), C.c_void_p(out_regress.data_ptr()),
                                       C.c_void_p(out_binary.data_ptr()), _stream_ptr(stream)))
            return out_logits, out_regress, out_binary
        if out_logits is None:
            out_logits = torch.empty((N, self.n_classes), dtype=torch.float32, device=elements.device)
        if out_regress is None:
            out_regress = torch.empty((N, self.n_regress), dtype=torch.float32, device=elements.device)
        _check(lib().mlpf_infer(self._h, C.c_void_p(elements.data_ptr()), off.ctypes.data_as(C.c_void_p),
                                len(off) - 1, C.c_void_p(out_logits.data_ptr()),
                                C.c_void_p(out_regress.data_ptr()), _stream_ptr(stream)))
        return out_logits, out_regress

    def infer_host(self, elements_host, event_offsets, out_logits_host, out_regress_host, stream=None):
        """Host (ideally pinned) torch tensors in and out; copies + compute + synchronise inside."""
        off = np.ascontiguousarray(event_offsets, dtype=np.int32)
        _check(lib().mlpf_infer_host(self._h, C.c_void_p(elements_host.data_ptr()),
                                     off.ctypes.data_as(C.c_void_p), len(off) - 1,
                                     C.c_void_p(out_logits_host.data_ptr()),
                                     C.c_void_p(out_regress_host.data_ptr()), _stream_ptr(stream)))

    def infer_host_async(self, elements_host, event_offsets, out_logits_host, out_regress_host, stream=None):
        """As infer_host without the final synchronisation (call host_sync before reading the outputs)."""
        off = np.ascontiguousarray(event_offsets, dtype=np.int32)
        _check(lib().mlpf_infer_host_async(self._h, C.c_void_p(elements_host.data_ptr()),
                                           off.ctypes.data_as(C.c_void_p), len(off) - 1,
                                           C.c_void_p(out_logits_host.data_ptr()),
                                           C.c_void_p(out_regress_host.data_ptr()), _stream_ptr(stream)))

    def host_sync(self, stream=None):
        _check(lib().mlpf_host_sync(self._h, _stream_ptr(stream)))

    def schedule(self, which: str, stream=None):
        cap = 1 << 22
        out = np.empty(cap, np.int32)
        n = _check(lib().mlpf_debug_get_schedule(self._h, _stream_ptr(stream), SCHED[which],
                                                 out.ctypes.data_as(C.c_void_p), cap))
        out = out[:n].copy()
        return out.reshape(-1, 2) if which == "work_list" else out

    def profile(self, stream=None):
        """{kernel class: (ms, launches)} of the last infer on `stream` (needs OPT_PROFILE = 1)."""
        ms = (C.c_float * len(KERNEL_CLASSES))()
        cnt = (C.c_int32 * len(KERNEL_CLASSES))()
        _check(lib().mlpf_debug_get_profile(self._h, _stream_ptr(stream), ms, cnt))
        return {k: (float(ms[i]), int(cnt[i])) for i, k in enumerate(KERNEL_CLASSES)}

    def tensor(self, which: str, shape, stream=None):
        out = np.empty(int(np.prod(shape)), np.float32)
        n = _check(lib().mlpf_debug_get_tensor(self._h, _stream_ptr(stream), TENSOR[which],
                                               out.ctypes.data_as(C.c_void_p), out.size))
        assert n == out.size, (n, out.size)
        return out.reshape(shape)


def tc_gemm_bf16(A, W, A_lo=None, stream=None):
    """A (+ A_lo) [M,K], W [N,K] CUDA bfloat16 tensors -> fp32 [M,N] = (A + A_lo) W^T via the tcgen05 GEMM."""
    import torch
    M, K = A.shape
    N = W.shape[0]
    out = torch.empty((M, N), dtype=torch.float32, device=A.device)
    _check(lib().mlpf_tc_gemm_bf16(C.c_void_p(A.data_ptr()), C.c_void_p(A_lo.data_ptr() if A_lo is not None else 0),
                                   C.c_void_p(W.data_ptr()), C.c_void_p(out.data_ptr()),
                                   M, N, K, _stream_ptr(stream)))
    return out


def tc_attention_bf16(QKV, key_valid, event_offsets, d_model, n_heads, stream=None, impl=1):
    """QKV [N,3d] bf16 (q | k | v), key_valid [N] int32 or None -> O [N,d] bf16 (Eq. 4 per event/head).
    impl: 1 = bound-based kernel (default), 2 = its exact path forced, 0 = round 1's lazy-rescale kernel; 3 / 4 = 1 / 2
    for a QKV whose q columns already carry the factor log2(e) / sqrt(head_dim)."""
    import torch
    _check(lib().mlpf_debug_set_attention_impl(int(impl)))
    off = np.ascontiguousarray(event_offsets, dtype=np.int32)
    assert QKV.is_contiguous() and QKV.shape[1] == 3 * d_model
    N = QKV.shape[0]
    out = torch.zeros((N, d_model), dtype=torch.bfloat16, device=QKV.device)
    kv = C.c_void_p(key_valid.data_ptr()) if key_valid is not None else C.c_void_p(0)
    _check(lib().mlpf_tc_attention_bf16(C.c_void_p(QKV.data_ptr()), kv,
                                        off.ctypes.data_as(C.c_void_p), len(off) - 1, d_model, n_heads,
                                        C.c_void_p(out.data_ptr()), _stream_ptr(stream)))
    return out


def tc_gemm_fp8(A8, W8, out_scale=1.0, stream=None):
    """A8 [M,K], W8 [N,K] CUDA tensors of dtype float8_e4m3fn -> fp32 [M,N] = out_scale * A W^T via the tcgen05 f8f6f4 GEMM."""
    import torch
    M, K = A8.shape
    N = W8.shape[0]
    out = torch.empty((M, N), dtype=torch.float32, device=A8.device)
    _check(lib().mlpf_tc_gemm_fp8(C.c_void_p(A8.data_ptr()), C.c_void_p(W8.data_ptr()), C.c_void_p(out.data_ptr()),
                                  M, N, K, float(out_scale), _stream_ptr(stream)))
    return out


def microbench(which, iters=2048, stream=None):
    """results per clock per SM: 0 ex2.f32 (MUFU), 1 ex2.bf16x2 (MUFU), 2 polynomial 2^x (FMA/ALU), 3 fma.f32x2 pairs."""
    r = lib().mlpf_microbench(int(which), int(iters), _stream_ptr(stream))
    if r < 0:
        raise MlpfError("mlpf_microbench: " + lib().mlpf_last_error().decode())
    return float(r)


def tc_post_bf16(o_hi, o_lo, h, Wo, bo, ln2g, ln2b, W1, b1, W2, b2, lnng, lnnb, activation, eps, want_lo=True, stream=None):
    """The fused post-attention block (include/mlpf.h mlpf_tc_post_bf16).  CUDA tensors: o_hi / o_lo [M,d] bf16, h [M,d]
    fp32 (updated in place), weights bf16 [out,in], vectors fp32 (lnng / lnnb may be None).  Returns (u_hi, u_lo)."""
    import torch
    M, d = h.shape
    dff = W1.shape[0]
    u_hi = torch.empty((M, d), dtype=torch.bfloat16, device=h.device)
    u_lo = torch.empty((M, d), dtype=torch.bfloat16, device=h.device) if want_lo else None
    ptr = lambda t: C.c_void_p(t.data_ptr() if t is not None else 0)
    _check(lib().mlpf_tc_post_bf16(ptr(o_hi), ptr(o_lo), ptr(h), ptr(Wo), ptr(bo), ptr(ln2g), ptr(ln2b), ptr(W1), ptr(b1),
                                   ptr(W2), ptr(b2), ptr(lnng), ptr(lnnb), M, d, dff, int(activation), float(eps),
                                   ptr(u_hi), ptr(u_lo), _stream_ptr(stream)))
    return u_hi, u_lo


def build_candidates(elements, event_offsets, logits, regress, scratch=None, stream=None, binary=None):
    """Per-event particle candidates from mlpf_infer's outputs (include/mlpf.h "candidate building").
    CUDA tensors in; returns dict(cand_offsets [E+1] int32, cand_elem [N] int32, cand_pid [N] int32,
    cand_p4 [N,4] float32 = (pT, eta, phi, E)), all CUDA, enqueued on `stream`; the first cand_offsets[-1]
    entries of the last three are the candidates."""
    import torch
    off = np.ascontiguousarray(event_offsets, dtype=np.int32)
    E = len(off) - 1
    N = int(off[-1]) if E >= 0 else 0
    dev = elements.device
    for t in (elements, logits, regress):
        assert t.is_cuda and t.dtype == torch.float32 and t.is_contiguous()
    assert regress.shape[1] == 5
    need = _check(lib().mlpf_candidates_scratch_bytes(N, max(E, 0)))
    if scratch is None:
        scratch = torch.empty(need, dtype=torch.uint8, device=dev)
    out = dict(cand_offsets=torch.empty(E + 1, dtype=torch.int32, device=dev),
               cand_elem=torch.empty(N, dtype=torch.int32, device=dev),
               cand_pid=torch.empty(N, dtype=torch.int32, device=dev),
               cand_p4=torch.empty((N, 4), dtype=torch.float32, device=dev))
    _check(lib().mlpf_build_candidates_ex(C.c_void_p(elements.data_ptr()), elements.shape[1], off.ctypes.data_as(C.c_void_p), E,
                                       C.c_void_p(logits.data_ptr()), logits.shape[1], C.c_void_p(regress.data_ptr()), regress.shape[1],
                                       C.c_void_p(binary.data_ptr() if binary is not None else 0),
                                       C.c_void_p(scratch.data_ptr()), scratch.numel(),
                                       C.c_void_p(out["cand_offsets"].data_ptr()), C.c_void_p(out["cand_elem"].data_ptr()),
                                       C.c_void_p(out["cand_pid"].data_ptr()), C.c_void_p(out["cand_p4"].data_ptr()),
                                       _stream_ptr(stream)))
    return out


def candidates_static_limit(which):
    """0: max elements per call, 1: max events per call, 2: bytes of device memory the library holds per GPU."""
    return _check(lib().mlpf_candidates_static_limit(which))


def build_candidates_static(elements, event_offsets, logits, regress, out, stream=None, binary=None):
    """mlpf_build_candidates_static: build_candidates without any allocation: the kernels' scratch is a device array
    inside the library and `out` is the caller's dict of preallocated CUDA tensors (cand_offsets [E+1] int32, cand_elem [N]
    int32, cand_pid [N] int32, cand_p4 [N,4] float32).  Calls that overlap on the GPU race on the shared scratch."""
    off = np.ascontiguousarray(event_offsets, dtype=np.int32)
    E = len(off) - 1
    _check(lib().mlpf_build_candidates_static(C.c_void_p(elements.data_ptr()), elements.shape[1], off.ctypes.data_as(C.c_void_p), E,
                                           C.c_void_p(logits.data_ptr()), logits.shape[1], C.c_void_p(regress.data_ptr()), regress.shape[1],
                                           C.c_void_p(binary.data_ptr() if binary is not None else 0),
                                           C.c_void_p(out["cand_offsets"].data_ptr()), C.c_void_p(out["cand_elem"].data_ptr()),
                                           C.c_void_p(out["cand_pid"].data_ptr()), C.c_void_p(out["cand_p4"].data_ptr()),
                                           _stream_ptr(stream)))
    return out
