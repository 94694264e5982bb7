"""CPU oracle for the H-HIGNN hot path -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Thin ctypes wrapper over oracle/hh_oracle.cpp (plain fp64 C++ written from PAPER.md).  Only
tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this package.  It imports nothing from paper_2505_08174_b200 and shares no code with it.
"""
import ctypes as C
import numpy as np
from . import build as _build

_lib = None

_f32p = np.ctypeslib.ndpointer(np.float32, flags="C_CONTIGUOUS")
_f64p = np.ctypeslib.ndpointer(np.float64, flags="C_CONTIGUOUS")
_i32p = np.ctypeslib.ndpointer(np.int32, flags="C_CONTIGUOUS")
_i64p = np.ctypeslib.ndpointer(np.int64, flags="C_CONTIGUOUS")
_u64p = np.ctypeslib.ndpointer(np.uint64, flags="C_CONTIGUOUS")


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build.build())
        _lib.orc_h_create.restype = C.c_void_p
        _lib.orc_h_matvec.restype = C.c_int64
        _lib.orc_h_aca_block.restype = C.c_int
        _lib.orc_num_threads.restype = C.c_int
        _lib.orc_h_admissible.restype = C.c_int
        _lib.orc_h_last_bad_strict.restype = C.c_int64
    return _lib


def num_threads():
    return int(lib().orc_num_threads())


def pack_mlp(Ws, bs):
    """(dims int32[nl+1], nl, flat fp32 params W0,b0,W1,b1,...) from lists of [out][in] weights."""
    dims = [Ws[0].shape[1]] + [W.shape[0] for W in Ws]
    flat = np.concatenate([np.concatenate([np.ascontiguousarray(W, np.float32).ravel(),
                                           np.ascontiguousarray(b, np.float32).ravel()])
                           for W, b in zip(Ws, bs)]).astype(np.float32)
    return np.asarray(dims, np.int32), len(Ws), flat


def _vp(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def mlp_forward(mlp, x):
    dims, nl, flat = pack_mlp(*mlp)
    x = np.ascontiguousarray(x, np.float64)
    y = np.zeros(int(dims[-1]), np.float64)
    lib().orc_mlp_forward(_vp(dims), nl, _vp(flat), _vp(x), _vp(y))
    return y


def entry2(mlp, a, Xi, Xj):
    dims, nl, flat = pack_mlp(*mlp)
    Xi = np.ascontiguousarray(Xi, np.float32)
    Xj = np.ascontiguousarray(Xj, np.float32)
    M = np.zeros(9, np.float64)
    lib().orc_entry2(_vp(dims), nl, _vp(flat), C.c_double(a), _vp(Xi), _vp(Xj), _vp(M))
    return M.reshape(3, 3)


def dense_matvec(X, F, mlp, a=1.0, include_self=True, rows=None):
    dims, nl, flat = pack_mlp(*mlp)
    X = np.ascontiguousarray(X, np.float32)
    F = np.ascontiguousarray(F, np.float32)
    N = X.shape[0]
    if rows is None:
        U = np.zeros((N, 3), np.float64)
        lib().orc_dense_matvec(C.c_int64(N), _vp(X), _vp(F), _vp(dims), nl, _vp(flat), C.c_double(a),
                               int(include_self), _vp(U))
        return U
    rows = np.ascontiguousarray(rows, np.int64)
    U = np.zeros((len(rows), 3), np.float64)
    lib().orc_dense_rows(C.c_int64(N), _vp(X), _vp(F), _vp(dims), nl, _vp(flat), C.c_double(a),
                         int(include_self), C.c_int64(len(rows)), _vp(rows), _vp(U))
    return U


def three_body(X, F, mlp3, rcut, brute=False):
    """Three-body term only (no self, no two-body). Returns (U, n_faces)."""
    dims, nl, flat = pack_mlp(*mlp3)
    X = np.ascontiguousarray(X, np.float32)
    F = np.ascontiguousarray(F, np.float32)
    N = X.shape[0]
    U = np.zeros((N, 3), np.float64)
    nf = C.c_int64(0)
    fn = lib().orc_three_body_brute if brute else lib().orc_three_body
    fn(C.c_int64(N), _vp(X), _vp(F), _vp(dims), nl, _vp(flat), C.c_float(rcut), _vp(U), C.byref(nf))
    return U, int(nf.value)


def self_terms(X, F, mlp2, mlp3, rcut, a=1.0):
    """The diagonal terms M^(s,2) F + M^(s,3) F of Eq. (6) from the self halves (first 9 outputs) of
    18-output networks; a network with 9 outputs (or None) contributes nothing.  Returns (U, n_pairs, n_faces)."""
    X = np.ascontiguousarray(X, np.float32)
    F = np.ascontiguousarray(F, np.float32)
    N = X.shape[0]
    U = np.zeros((N, 3), np.float64)
    d2, n2, f2 = pack_mlp(*mlp2) if mlp2 is not None else (None, 0, None)
    d3, n3, f3 = pack_mlp(*mlp3) if mlp3 is not None else (None, 0, None)
    npairs, nf = C.c_int64(0), C.c_int64(0)
    lib().orc_self_terms(C.c_int64(N), _vp(X), _vp(F), _vp(d2), n2, _vp(f2), _vp(d3), n3, _vp(f3), C.c_double(a), C.c_float(rcut),
                         _vp(U), C.byref(npairs), C.byref(nf))
    return U, int(npairs.value), int(nf.value)


def morton_keys(X):
    X = np.ascontiguousarray(X, np.float32)
    keys = np.zeros(X.shape[0], np.uint64)
    lib().orc_morton_keys(C.c_int64(X.shape[0]), _vp(X), _vp(keys))
    return keys


def euler(X, U, dt):
    X = np.array(X, np.float32, copy=True, order="C")
    U = np.ascontiguousarray(U, np.float64)
    lib().orc_euler(C.c_int64(X.shape[0]), _vp(X), _vp(U), C.c_float(dt))
    return X


class HMatrix:
    """O-H: cluster tree + Alg. 1 block lists for (X, leaf, eta), ACA and the H mat-vec."""

    def __init__(self, X, mlp2, leaf=64, eta=1.0, a=1.0):
        self.X = np.ascontiguousarray(X, np.float32)
        self.N = self.X.shape[0]
        dims, nl, flat = pack_mlp(*mlp2)
        self._h = C.c_void_p(lib().orc_h_create(C.c_int64(self.N), _vp(self.X), int(leaf), C.c_double(eta),
                                                _vp(dims), nl, _vp(flat), C.c_double(a)))
        c = [C.c_int64(0) for _ in range(5)]
        lib().orc_h_counts(self._h, *[C.byref(v) for v in c])
        self.n_nodes, self.n_leaves, self.nG, self.nH, self.depth = [int(v.value) for v in c]
        n = self.n_nodes
        self.perm = np.zeros(self.N, np.int64)
        self.keys = np.zeros(self.N, np.uint64)
        self.lo = np.zeros(n, np.int64)
        self.hi = np.zeros(n, np.int64)
        self.left = np.zeros(n, np.int32)
        self.right = np.zeros(n, np.int32)
        self.parent = np.zeros(n, np.int32)
        self.level = np.zeros(n, np.int32)
        self.bmin = np.zeros((n, 3), np.float32)
        self.bmax = np.zeros((n, 3), np.float32)
        lib().orc_h_get_tree(self._h, _vp(self.perm), _vp(self.keys), _vp(self.lo), _vp(self.hi), _vp(self.left),
                             _vp(self.right), _vp(self.parent), _vp(self.level), _vp(self.bmin), _vp(self.bmax))
        self.G = np.zeros((self.nG, 2), np.int32)
        self.H = np.zeros((self.nH, 2), np.int32)
        for which, arr in ((0, self.G), (1, self.H)):
            t = np.zeros(len(arr), np.int32)
            s = np.zeros(len(arr), np.int32)
            lib().orc_h_get_blocks(self._h, which, _vp(t), _vp(s))
            arr[:, 0], arr[:, 1] = t, s

    def set_replay_roundoff(self, u):
        """Replay checker only: unit roundoff of the arithmetic being replayed (2**-24 for the fp32 CUDA
        path).  A replayed pivot / stop decision then counts as bad only if it is outside the slack AND
        outside the running rounding bound of that arithmetic (arg-max "up to rounding")."""
        lib().orc_h_set_replay_roundoff(self._h, C.c_double(u))

    def set_kappa_max(self, kappa):
        """S-18b: pivot blocks with cond_F = |P|_F |P^-1|_F above kappa break Alg. 2 down (flag 2, block applied
        densely).  Opt-in: the default is float('inf'), the listing as printed."""
        lib().orc_h_set_kappa_max(self._h, C.c_double(kappa))

    def set_dense_cap(self, cap):
        """S-18b applies to blocks with |tau||sigma| <= cap (|tau| + |sigma|) only (default 128)."""
        lib().orc_h_set_dense_cap(self._h, C.c_double(cap))

    def last_bad_strict(self):
        """slack-only count of bad decisions of the last replay call (reported, not asserted)"""
        return int(lib().orc_h_last_bad_strict(self._h))

    def __del__(self):
        try:
            lib().orc_h_destroy(self._h)
        except Exception:
            pass

    # ---- comparisons use ranges, not node numbering (S-12, S-16) ----
    def node_table(self):
        """sorted rows (lo, hi, is_leaf) + boxes in the same order"""
        order = np.lexsort((self.hi, self.lo))
        return (np.stack([self.lo, self.hi, (self.left < 0).astype(np.int64)], 1)[order],
                self.bmin[order], self.bmax[order])

    def block_table(self, which):
        """sorted rows (tau_lo, tau_hi, sigma_lo, sigma_hi) of P^G ('G') or P^H ('H')"""
        B = self.G if which == "G" else self.H
        T = np.stack([self.lo[B[:, 0]], self.hi[B[:, 0]], self.lo[B[:, 1]], self.hi[B[:, 1]]], 1)
        return T[np.lexsort((T[:, 3], T[:, 2], T[:, 1], T[:, 0]))] if len(T) else T.reshape(0, 4)

    def admissible(self, t, s):
        return bool(lib().orc_h_admissible(self._h, int(t), int(s)))

    def block_shape(self, g):
        t, s = self.G[g]
        return int(self.hi[t] - self.lo[t]), int(self.hi[s] - self.lo[s])

    def aca_block(self, g, zeta, max_rank=96, rule=0, replay=None, slack=1e-3, replay_flag=0):
        """Alg. 2 on admissible block g. replay=(piv_i, piv_j) re-runs with given pivots/rank; with replay_flag=2
        the last pivot pair is the attempted one at which the replayed run broke down (S-18b).
        Returns dict(rank, C[l,c,3,3], Q[l,q,3,3], piv_i, piv_j, nu, lam, flag, replay_bad)."""
        c, q = self.block_shape(g)
        cap = min(c, q, max_rank) + 1
        Cb = np.zeros((cap, c, 3, 3), np.float64)
        Qb = np.zeros((cap, q, 3, 3), np.float64)
        pi = np.zeros(cap, np.int32)
        pj = np.zeros(cap, np.int32)
        nu = np.zeros(cap, np.float64)
        lam = np.zeros(cap, np.float64)
        flag = C.c_int(0)
        bad = C.c_int(0)
        if replay is None:
            rr, ri, rj = -1, None, None
        else:
            ri = np.ascontiguousarray(replay[0], np.int32)
            rj = np.ascontiguousarray(replay[1], np.int32)
            rr = len(ri) - (1 if replay_flag == 2 else 0)
        r = lib().orc_h_aca_block(self._h, C.c_int64(g), C.c_double(zeta), int(max_rank), int(rule), int(rr),
                                  int(replay_flag), _vp(ri), _vp(rj), C.c_double(slack), int(cap), _vp(Cb), _vp(Qb), _vp(pi),
                                  _vp(pj), _vp(nu), _vp(lam), C.byref(flag), C.byref(bad))
        npiv = r + (1 if int(flag.value) == 2 and r < cap else 0)       # a breakdown also lists its attempted pivot
        return dict(rank=r, C=Cb[:r], Q=Qb[:r], piv_i=pi[:npiv], piv_j=pj[:npiv], nu=nu[:r], lam=lam[:r],
                    flag=int(flag.value), replay_bad=int(bad.value))

    def dense_block(self, g):
        c, q = self.block_shape(g)
        G = np.zeros((c, q, 3, 3), np.float64)
        lib().orc_h_dense_block(self._h, C.c_int64(g), _vp(G))
        return G

    def matvec(self, F, zeta, max_rank=96, rule=0, include_self=True, near=True, far=True,
               replay=None, slack=1e-3, only_rows=None):
        """U = M_H(X) F in caller order. replay = (ranks[nG], piv_i concat, piv_j concat[, flags[nG]]) in THIS
        object's P^G order; a block with flag 2 lists ranks[g] + 1 pivot pairs (the last one is the attempted
        pivot at which the replayed run broke down, S-18b).  Returns (U, info)."""
        F = np.ascontiguousarray(F, np.float32)
        U = np.zeros((self.N, 3), np.float64)
        ranks = np.zeros(self.nG, np.int32)
        flags = np.zeros(self.nG, np.int32)
        ne = C.c_int64(0)
        if replay is None:
            rr = rf = ro = ri = rj = None
        else:
            rr = np.ascontiguousarray(replay[0], np.int32)
            rf = np.ascontiguousarray(replay[3], np.int32) if len(replay) > 3 else np.zeros(self.nG, np.int32)
            ro = np.zeros(self.nG, np.int64)
            if self.nG:
                ro[1:] = np.cumsum((rr + (rf == 2))[:-1])
            ri = np.ascontiguousarray(replay[1], np.int32)
            rj = np.ascontiguousarray(replay[2], np.int32)
        rows = None if only_rows is None else np.ascontiguousarray(only_rows, np.uint8)
        bad = lib().orc_h_matvec(self._h, _vp(F), C.c_double(zeta), int(max_rank), int(rule), int(include_self),
                                 int(near), int(far), _vp(rr), _vp(rf), _vp(ro), _vp(ri), _vp(rj), C.c_double(slack),
                                 _vp(rows), _vp(U), _vp(ranks), _vp(flags), C.byref(ne))
        return U, dict(ranks=ranks, flags=flags, entries=int(ne.value), replay_bad=int(bad))
