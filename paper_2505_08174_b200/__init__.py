"""paper_2505_08174_b200 -- thin Python binding of the C ABI in include/hh.h (libhh.so).

Argument marshalling only: every step of the hot path (tree, block partition, ACA, near-/far-field
apply, three-body term, Euler step) runs in the CUDA kernels under csrc/.  PyTorch is used for device
memory and streams.  There is no CPU fallback: without the compiled library or without a CUDA device
the calls raise.
"""
import ctypes as C
import os

import numpy as np

from . import build as _build

_HERE = os.path.dirname(os.path.abspath(__file__))
_lib = None

HH_OK = 0
ERRORS = {-1: "HH_ERR_INVALID_ARG", -2: "HH_ERR_WORKSPACE_TOO_SMALL", -3: "HH_ERR_CUDA", -4: "HH_ERR_NOT_BUILT",
          -5: "HH_ERR_UNSUPPORTED"}

EXPORTS = ["hh_create", "hh_destroy", "hh_set_params", "hh_enable_timing", "hh_build_tree", "hh_build_blocks", "hh_aca",
           "hh_matvec", "hh_matvec_parts", "hh_set_aca_impl", "hh_set_far_impl", "hh_far_apply_resident", "hh_step", "hh_step_host", "hh_set_pair_capacity",
           "hh_get_stats", "hh_get_tree", "hh_get_blocks", "hh_get_factors", "hh_get_ranks", "hh_eval_entries",
           "hh_set_capture", "hh_get_capture_count", "hh_last_error", "hh_version", "hh_dense_matvec_static"]


class HHError(RuntimeError):
    def __init__(self, code, text):
        super().__init__("%s (%d): %s" % (ERRORS.get(code, "?"), code, text))
        self.code = code


class _Mlp(C.Structure):
    _fields_ = [("n_layers", C.c_int32), ("dims", C.POINTER(C.c_int32)), ("W", C.POINTER(C.c_void_p)),
                ("b", C.POINTER(C.c_void_p))]


class _Params(C.Structure):
    _fields_ = [("leaf_size", C.c_int32), ("eta", C.c_float), ("aca_tol", C.c_float), ("aca_max_rank", C.c_int32),
                ("radius_a", C.c_float), ("rcut3", C.c_float), ("pivot_rule", C.c_int32), ("near_path", C.c_int32),
                ("kappa_max", C.c_float), ("dense_cap", C.c_float), ("aca_precision", C.c_int32)]


class Stats(C.Structure):
    _fields_ = [(n, C.c_int64) for n in
                ("n_particles", "n_nodes", "n_leaves", "depth", "n_admissible", "n_inadmissible", "near_entries",
                 "far_rows_cols", "sum_rank", "aca_entries", "factor_bytes", "aca_batches", "aca_not_converged",
                 "aca_singular", "n_faces", "workspace_required", "arena_bytes")] + \
               [(n, C.c_float) for n in ("ms_tree", "ms_blocks", "ms_aca", "ms_near", "ms_far", "ms_three", "ms_other", "pad_")] + \
               [("n_launches", C.c_int64), ("fallback_entries", C.c_int64), ("n_self_pairs", C.c_int64)]

    def as_dict(self):
        return {n: getattr(self, n) for n, _ in self._fields_}


def lib_path():
    return os.environ.get("HH_LIB_PATH") or os.path.join(_HERE, "libhh.so")      # HH_LIB_PATH: try another build of the same ABI


def load(build_if_missing=True):
    """Load libhh.so (building it in-tree first if it is missing).  Raises if it cannot be had."""
    global _lib
    if _lib is None:
        p = lib_path()
        if not os.path.exists(p):
            if not build_if_missing:
                raise RuntimeError("libhh.so is missing: run python -m paper_2505_08174_b200.build")
            _build.build()
        _lib = C.CDLL(p)
        _lib.hh_last_error.restype = C.c_char_p
        _lib.hh_version.restype = C.c_char_p
    return _lib


def _ptr(t):
    """device (torch) or host (numpy) pointer as void*; None -> NULL"""
    if t is None:
        return None
    if isinstance(t, np.ndarray):
        assert t.flags["C_CONTIGUOUS"]
        return C.c_void_p(t.ctypes.data)
    assert t.is_contiguous()
    return C.c_void_p(t.data_ptr())


STATIC_MAX_N = 16384                      # HH_STATIC_MAX_N of include/hh.h


class DeviceMlp:
    """An hh_mlp whose layers live on the device (torch tensors owned here): the argument of dense_matvec_static"""

    def __init__(self, mlp, device="cuda:0"):
        import torch
        Ws, bs = mlp
        self.dims = (C.c_int32 * (len(Ws) + 1))(*([Ws[0].shape[1]] + [W.shape[0] for W in Ws]))
        self.W = [torch.from_numpy(np.ascontiguousarray(W, np.float32)).to(device) for W in Ws]
        self.b = [torch.from_numpy(np.ascontiguousarray(b, np.float32)).to(device) for b in bs]
        self.pW = (C.c_void_p * len(Ws))(*[t.data_ptr() for t in self.W])
        self.pb = (C.c_void_p * len(bs))(*[t.data_ptr() for t in self.b])
        self.struct = _Mlp(len(Ws), self.dims, self.pW, self.pb)


def dense_matvec_static(dmlp, X, F, radius_a=1.0, out=None, stream=None):
    """hh_dense_matvec_static: the entry point that allocates nothing (static device scratch, N <= STATIC_MAX_N).
    X, F: torch CUDA fp32 [N][3]; `out` (same shape) is overwritten, or a new tensor is returned (that allocation is
    the binding's, not the library's).  Argument marshalling only."""
    import torch
    lib = load()
    if not torch.cuda.is_available():
        raise RuntimeError("paper_2505_08174_b200 needs a CUDA device (there is no CPU fallback)")
    U = out if out is not None else torch.empty_like(F)
    st = stream if stream is not None else torch.cuda.current_stream(X.device)
    err = C.create_string_buffer(512)
    r = lib.hh_dense_matvec_static(C.byref(dmlp.struct), C.c_float(radius_a), _ptr(X), _ptr(F), _ptr(U), C.c_int64(X.shape[0]),
                                   C.c_void_p(st.cuda_stream), err, C.c_size_t(512))
    if r != HH_OK:
        raise HHError(r, err.value.decode())
    return U


class Context:
    """One hh_ctx.  `mlp2` / `mlp3` are (Ws, bs) lists of numpy arrays ([out][in] weights); the
    workspace is a torch uint8 CUDA tensor owned here (PyTorch owns all device memory)."""

    def __init__(self, mlp2, mlp3=None, leaf_size=64, eta=1.0, aca_tol=1e-4, aca_max_rank=96, radius_a=1.0, rcut3=0.0,
                 pivot_rule=0, near_path=0, kappa_max=0.0, dense_cap=0.0, aca_precision=0, workspace_bytes=None, device="cuda:0", stream=None):
        import torch
        self.torch = torch
        self.lib = load()
        if not torch.cuda.is_available():
            raise RuntimeError("paper_2505_08174_b200 needs a CUDA device (there is no CPU fallback)")
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        if workspace_bytes is None:
            free, _ = torch.cuda.mem_get_info(self.device)
            workspace_bytes = int(free * 0.80)
        self.workspace = torch.empty(int(workspace_bytes) // 256 * 256, dtype=torch.uint8, device=self.device)
        self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        self._keep = []
        self.params = _Params(leaf_size, eta, aca_tol, aca_max_rank, radius_a, rcut3, pivot_rule, near_path, kappa_max, dense_cap, aca_precision)
        m2 = self._mlp_struct(mlp2)
        m3 = self._mlp_struct(mlp3) if mlp3 is not None else None
        self._h = C.c_void_p()
        r = self.lib.hh_create(C.byref(self._h), C.byref(self.params), C.byref(m2), C.byref(m3) if m3 else None,
                               _ptr(self.workspace), C.c_size_t(self.workspace.numel()), C.c_void_p(self.stream.cuda_stream))
        if r != HH_OK:
            text = self.lib.hh_last_error(self._h).decode() if self._h else "hh_create failed"
            if self._h:
                self.lib.hh_destroy(self._h)
                self._h = C.c_void_p()
            raise HHError(r, text)
        self.N = 0

    def _mlp_struct(self, mlp):
        torch = self.torch
        Ws, bs = mlp
        dims = (C.c_int32 * (len(Ws) + 1))(*([Ws[0].shape[1]] + [W.shape[0] for W in Ws]))
        dW = [torch.from_numpy(np.ascontiguousarray(W, np.float32)).to(self.device) for W in Ws]
        db = [torch.from_numpy(np.ascontiguousarray(b, np.float32)).to(self.device) for b in bs]
        pW = (C.c_void_p * len(Ws))(*[t.data_ptr() for t in dW])
        pb = (C.c_void_p * len(bs))(*[t.data_ptr() for t in db])
        self._keep += [dims, dW, db, pW, pb]
        return _Mlp(len(Ws), dims, pW, pb)

    def _chk(self, r):
        if r != HH_OK:
            raise HHError(r, self.lib.hh_last_error(self._h).decode())

    def close(self):
        if getattr(self, "_h", None):
            self.lib.hh_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- the hot path: same names as the C ABI ----
    def set_params(self, **kw):
        for k, v in kw.items():
            setattr(self.params, k, v)
        self._chk(self.lib.hh_set_params(self._h, C.byref(self.params)))

    def set_pair_capacity(self, pairs_per_particle):
        self._chk(self.lib.hh_set_pair_capacity(self._h, C.c_int64(pairs_per_particle)))

    def set_aca_impl(self, impl):
        self._chk(self.lib.hh_set_aca_impl(self._h, int(impl)))

    def set_far_impl(self, impl):
        self._chk(self.lib.hh_set_far_impl(self._h, int(impl)))

    def enable_timing(self, on=True):
        self._chk(self.lib.hh_enable_timing(self._h, int(on)))

    def build_tree(self, X):
        self.N = int(X.shape[0])
        self._chk(self.lib.hh_build_tree(self._h, _ptr(X), C.c_int64(self.N)))

    def build_blocks(self):
        self._chk(self.lib.hh_build_blocks(self._h))

    def aca(self, first_block=0):
        nxt = C.c_int64(0)
        self._chk(self.lib.hh_aca(self._h, C.c_int64(first_block), C.byref(nxt)))
        return int(nxt.value)

    def matvec(self, F, U=None, parts=31):
        if U is None:
            U = self.torch.empty_like(F)
        self._chk(self.lib.hh_matvec_parts(self._h, _ptr(F), _ptr(U), int(parts)))
        return U

    def far_apply_resident(self, F, U=None):
        if U is None:
            U = self.torch.empty_like(F)
        self._chk(self.lib.hh_far_apply_resident(self._h, _ptr(F), _ptr(U)))
        return U

    def step(self, X, F, U=None, dt=0.0):
        if U is None:
            U = self.torch.empty_like(F)
        self.N = int(X.shape[0])
        self._chk(self.lib.hh_step(self._h, _ptr(X), _ptr(F), _ptr(U), C.c_int64(self.N), C.c_float(dt)))
        return U

    def step_host(self, X, F, U, dt=0.0):
        """X, F, U: host arrays (numpy or pinned CPU torch tensors); X is updated in place."""
        self.N = int(X.shape[0])
        self._chk(self.lib.hh_step_host(self._h, _ptr(X), _ptr(F), _ptr(U), C.c_int64(self.N), C.c_float(dt)))
        return U

    def set_capture(self, row_prefix=None, records=None):
        """row_prefix: int32 CUDA tensor [N+1]; records: int32 CUDA tensor [cap][200]; both None = off (see hh.h)"""
        self._capture = (row_prefix, records)                            # keep the buffers alive
        cap = 0 if records is None else int(records.shape[0])
        self._chk(self.lib.hh_set_capture(self._h, _ptr(row_prefix), _ptr(records), C.c_int64(cap)))

    def capture_count(self):
        n = C.c_int64(0)
        self._chk(self.lib.hh_get_capture_count(self._h, C.byref(n)))
        return int(n.value)

    # ---- introspection ----
    def stats(self):
        st = Stats()
        self._chk(self.lib.hh_get_stats(self._h, C.byref(st)))
        return st.as_dict()

    def get_tree(self):
        st = self.stats()
        N, n = st["n_particles"], st["n_nodes"]
        out = dict(perm=np.zeros(N, np.int64), keys=np.zeros(N, np.uint64), lo=np.zeros(n, np.int64), hi=np.zeros(n, np.int64),
                   left=np.zeros(n, np.int32), right=np.zeros(n, np.int32), parent=np.zeros(n, np.int32),
                   level=np.zeros(n, np.int32), bmin=np.zeros((n, 3), np.float32), bmax=np.zeros((n, 3), np.float32))
        self._chk(self.lib.hh_get_tree(self._h, *[_ptr(out[k]) for k in
                                                   ("perm", "keys", "lo", "hi", "left", "right", "parent", "level", "bmin", "bmax")]))
        return out

    def get_blocks(self, which):
        st = self.stats()
        n = st["n_admissible"] if which in (0, "G") else st["n_inadmissible"]
        t, s = np.zeros(n, np.int32), np.zeros(n, np.int32)
        self._chk(self.lib.hh_get_blocks(self._h, 0 if which in (0, "G") else 1, _ptr(t), _ptr(s)))
        return t, s

    def get_ranks(self):
        n = self.stats()["n_admissible"]
        r, f = np.zeros(n, np.int32), np.zeros(n, np.int32)
        self._chk(self.lib.hh_get_ranks(self._h, _ptr(r), _ptr(f)))
        return r, f

    def get_factors(self, block, m, n, cap_rank=96, want_factors=True):
        rank, flag = C.c_int32(0), C.c_int32(0)
        pi, pj = np.zeros(cap_rank, np.int32), np.zeros(cap_rank, np.int32)
        Cf = np.zeros((cap_rank, m, 9), np.float32) if want_factors else None
        Qf = np.zeros((cap_rank, n, 9), np.float32) if want_factors else None
        self._chk(self.lib.hh_get_factors(self._h, C.c_int64(block), C.byref(rank), C.byref(flag), C.c_int32(cap_rank),
                                          _ptr(pi), _ptr(pj), _ptr(Cf), _ptr(Qf)))
        r = rank.value
        npiv = min(cap_rank, r + (1 if flag.value == 2 else 0))      # a breakdown also lists its attempted pivot
        return dict(rank=r, flag=flag.value, piv_i=pi[:npiv], piv_j=pj[:npiv], C=None if Cf is None else Cf[:r],
                    Q=None if Qf is None else Qf[:r])

    def eval_entries(self, Xi, Xj):
        M = self.torch.empty((Xi.shape[0], 9), dtype=self.torch.float32, device=self.device)
        self._chk(self.lib.hh_eval_entries(self._h, _ptr(Xi), _ptr(Xj), C.c_int64(Xi.shape[0]), _ptr(M)))
        return M
