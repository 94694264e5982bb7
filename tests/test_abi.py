"""The C-ABI library builds for sm_100a without a GPU, loads, and exports every symbol include/hh.h declares.
No compute call is made here (there is no GPU on this box); without a device hh_create must fail loudly."""
import ctypes as C
import os
import re

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "hh.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(hh_[a-z0-9_]+)\s*\(", text)))


def test_library_exports_every_declared_symbol():
    import paper_2505_08174_b200 as hh
    lib = C.CDLL(hh.build.build() if hasattr(hh, "build") else hh.lib_path())
    names = declared_symbols()
    assert {"hh_build_tree", "hh_build_blocks", "hh_aca", "hh_matvec", "hh_step"} <= set(names)   # the five BASELINE.json names
    missing = [n for n in names if not hasattr(lib, n)]
    assert not missing, missing
    assert set(names) <= set(hh.EXPORTS) | {"hh_ctx"}, sorted(set(names) - set(hh.EXPORTS))
    lib.hh_version.restype = C.c_char_p
    assert b"sm_100a" in lib.hh_version()


def test_params_struct_matches_header():
    import paper_2505_08174_b200 as hh
    text = open(os.path.join(ROOT, "include", "hh.h")).read()
    body = text[text.index("typedef struct {\n  int32_t leaf_size"):text.index("} hh_params;")]
    body = re.sub(r"/\*.*?\*/", "", body, flags=re.S)
    fields = re.findall(r"(?:int32_t|float)\s+([a-z_0-9]+)\s*;", body)
    assert fields == [n for n, _ in hh._Params._fields_]
    sbody = text[text.index("typedef struct {\n  int64_t n_particles"):text.index("} hh_stats;")]
    sbody = re.sub(r"/\*.*?\*/", "", sbody, flags=re.S)
    sfields = [f.strip() for decl in re.findall(r"(?:int64_t|float)\s+([^;]+);", sbody) for f in decl.split(",")]
    assert sfields == [n for n, _ in hh.Stats._fields_]


def test_no_cpu_fallback_without_a_device():
    import torch
    if torch.cuda.is_available():
        return                                    # on the GPU box the gpu-marked tests cover hh_create
    import paper_2505_08174_b200 as hh
    lib = hh.load()
    params = hh._Params(64, 1.0, 1e-4, 96, 1.0, 0.0, 0, 0, 0.0, 0.0)
    dims = (C.c_int32 * 4)(4, 32, 32, 9)
    pw = (C.c_void_p * 3)(0, 0, 0)
    mlp = hh._Mlp(3, dims, pw, pw)
    h = C.c_void_p()
    fake_ws = C.c_void_p(1 << 20)                 # aligned, never dereferenced: the device check comes first
    r = lib.hh_create(C.byref(h), C.byref(params), C.byref(mlp), None, fake_ws, C.c_size_t(1 << 30), None)
    assert r == -3 and not h.value               # HH_ERR_CUDA, no context
    try:
        hh.Context((None, None))
    except RuntimeError as e:
        assert "CUDA" in str(e)
    else:
        raise AssertionError("Context() must raise without a CUDA device")


def test_static_entry_point_checks_its_arguments_without_a_device():
    """hh_dense_matvec_static (the entry point that allocates nothing): size limit and argument errors come with a text before
    any CUDA call is made; with plausible arguments and no device it fails with HH_ERR_CUDA (no CPU fallback)."""
    import torch
    import paper_2505_08174_b200 as hh
    lib = hh.load()
    dims = (C.c_int32 * 4)(4, 32, 32, 9)
    one = C.c_void_p(256)                         # non-null, never dereferenced on these paths
    pw = (C.c_void_p * 3)(256, 256, 256)
    mlp = hh._Mlp(3, dims, pw, pw)
    err = C.create_string_buffer(256)

    def call(n, m=mlp, x=one):
        return lib.hh_dense_matvec_static(C.byref(m), C.c_float(1.0), x, one, one, C.c_int64(n), None, err, C.c_size_t(256))

    assert call(hh.STATIC_MAX_N + 1) == -2 and b"HH_STATIC_MAX_N" in err.value
    assert call(0) == -1 and b"N < 1" in err.value
    assert call(10, x=None) == -1
    bad = hh._Mlp(3, (C.c_int32 * 4)(7, 64, 64, 9), pw, pw)
    assert call(10, m=bad) == -5 and b"4-32-32-9" in err.value
    if not torch.cuda.is_available():
        assert call(10) == -3 and b"hh_dense_matvec_static" in err.value
