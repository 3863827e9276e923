"""CPU-side checks of the C-ABI boundary (no compute calls): the library builds, loads, exports every
symbol include/mlpf.h declares, and rejects malformed blobs before touching a device."""
import ctypes as C
import os
import re
import struct
import numpy as np
import pytest

import synth
import paper_2601_17554_b200 as P
from paper_2601_17554_b200 import build as B

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def L():
    B.build()
    return P.lib()


def test_library_exports_every_declared_symbol(L):
    hdr = open(os.path.join(ROOT, "include", "mlpf.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(mlpf_[a-z0-9_]+)\s*\(", hdr))
    assert {"mlpf_create", "mlpf_infer", "mlpf_destroy"} <= declared
    for name in declared:
        assert hasattr(L, name), name
    assert declared == set(P.EXPORTS)


def test_header_struct_matches_blob_writer():
    m = synth.model_cfg("cfg1")
    blob = P.pack_blob(synth.make_weights("cfg1"), m)
    assert len(blob) == 256 + 4 * synth.param_count(m)
    assert blob[:8] == b"MLPFBLOB"
    f = struct.unpack_from("<9I", blob, 8)
    assert f == (2, m.n_layers, m.d_model, m.n_heads, m.d_ff, 55, 4, 9, 4)
    assert struct.unpack_from("<2I", blob, 72) == (1, 0)                       # n_stacks, binary_head
    m2 = synth.model_cfg("paper2")
    blob2 = P.pack_blob(synth.make_weights("paper2"), m2)
    assert len(blob2) == 256 + 4 * synth.param_count(m2) and struct.unpack_from("<2I", blob2, 72) == (2, 1)
    assert struct.unpack_from("<4I", blob, 44) == (1, 1, 2, 1)
    assert struct.unpack_from("<2If", blob, 60)[:2] == (1, 1)


@pytest.mark.parametrize("mutate,needle", [
    (lambda b: b"XXXXXXXX" + b[8:], "magic"),
    (lambda b: b[:8] + struct.pack("<I", 7) + b[12:], "version"),
    (lambda b: b[:-4], "size"),
    (lambda b: b[:100], "header"),
    (lambda b: b[:16] + struct.pack("<I", 100) + b[20:], "hyper"),      # d_model = 100
])
def test_create_rejects_bad_blobs_before_touching_the_device(L, mutate, needle):
    m = synth.model_cfg("cfg1")
    blob = mutate(P.pack_blob(synth.make_weights("cfg1"), m))
    buf = C.create_string_buffer(blob, len(blob))
    h = L.mlpf_create(C.cast(buf, C.c_void_p), len(blob))
    assert not h
    assert needle in L.mlpf_last_error().decode()


def test_null_arguments(L):
    assert not L.mlpf_create(None, 0)
    assert L.mlpf_infer(None, None, None, 0, None, None, None) == -1
    assert L.mlpf_set_option(None, 1, 0) == -1
    assert L.mlpf_query(None, 1) == -1
    L.mlpf_destroy(None)


def test_no_cpu_fallback_without_a_device(L):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    with pytest.raises(P.MlpfError, match="no CUDA device"):
        P.Mlpf(synth.make_weights("cfg1"), synth.model_cfg("cfg1"))


def test_build_candidates_rejects_bad_arguments_before_touching_the_device(L):
    off = (C.c_int32 * 3)(0, 4, 2)
    assert L.mlpf_build_candidates(None, 55, off, 2, None, 9, None, None, 0, None, None, None, None, None) == -3
    assert "decreasing" in L.mlpf_last_error().decode()
    off = (C.c_int32 * 2)(1, 4)
    assert L.mlpf_build_candidates(None, 55, off, 1, None, 9, None, None, 0, None, None, None, None, None) == -3
    off = (C.c_int32 * 2)(0, 4)
    assert L.mlpf_build_candidates(None, 4, off, 1, None, 9, None, None, 0, None, None, None, None, None) == -6
    assert L.mlpf_build_candidates(None, 55, off, 1, None, 9, None, None, 0, None, None, None, None, None) == -1
    assert L.mlpf_build_candidates(None, 55, None, 0, None, 9, None, None, 0, None, None, None, None, None) == 0
    off = (C.c_int32 * 2)(0, 4)
    assert L.mlpf_build_candidates_ex(None, 55, off, 1, None, 9, None, 4, None, None, 0, None, None, None, None, None) == -6   # n_regress
    assert L.mlpf_build_candidates_ex(None, 55, off, 1, None, 49, None, 5, None, None, 0, None, None, None, None, None) == -6  # n_classes
    assert L.mlpf_candidates_scratch_bytes(1000, 4) >= 1000 + 5 * 4 + 2 * 4 * 4
    assert L.mlpf_candidates_scratch_bytes(-1, 0) < 0
