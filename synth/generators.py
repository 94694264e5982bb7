"""Synthetic suspensions shaped like the paper's workloads (§4)
and the five BASELINE.json configs.  Everything is drawn on the host from `rng.py`.

Stream ids: 0 positions, 1 (unused), 2 forces, 4 chain orientations; MLP weights use
their own seed (1 = two-body, 3 = three-body) with one stream per layer.
"""
import math
import numpy as np
from .rng import uniform01, normal01

MLP2_DIMS = (4, 32, 32, 9)    # two-body: [r_hat(3), a/r] -> 3x3   (BASELINE.json configs)
MLP3_DIMS = (7, 64, 64, 9)    # three-body: [r_ij(3), r_ik(3), |r_jk|] -> 3x3


# ----------------------------------------------------------------------------- positions
def cube_side(n, phi, a=1.0):
    return a * (n * 4.0 * math.pi / 3.0 / phi) ** (1.0 / 3.0)


def cube_cloud(n, phi, seed=0, a=1.0):
    """n i.i.d. uniform centres in a cube whose side gives volume fraction phi (C1, C3, C4)."""
    L = cube_side(n, phi, a)
    u = uniform01(seed, 0, 3 * n).reshape(n, 3)
    return (u * L).astype(np.float32)


def ball_cloud(n, phi, seed=0, a=1.0):
    """n centres uniform in a ball of radius a*(n/phi)^(1/3), by rejection from the cube,
    candidates taken in counter order (C2: spherical suspension drop)."""
    R = a * (n / phi) ** (1.0 / 3.0)
    out = np.empty((n, 3), dtype=np.float64)
    got, start = 0, 0
    while got < n:
        m = max(1024, int((n - got) * 2.2))
        u = uniform01(seed, 0, 3 * m, start=start).reshape(m, 3) * 2.0 - 1.0
        start += 3 * m
        keep = u[(u * u).sum(1) < 1.0]
        k = min(len(keep), n - got)
        out[got:got + k] = keep[:k]
        got += k
    return (out * R).astype(np.float32)


def chain_cloud(n_chains, n_beads, phi, bond=2.2, seed=0, a=1.0):
    """Straight bead chains, random orientation, centres uniform in a cube (C5)."""
    n = n_chains * n_beads
    L = cube_side(n, phi, a)
    c = uniform01(seed, 0, 3 * n_chains).reshape(n_chains, 3) * L
    z = uniform01(seed, 4, 2 * n_chains).reshape(n_chains, 2)
    cz = 2.0 * z[:, 0] - 1.0
    sz = np.sqrt(np.maximum(0.0, 1.0 - cz * cz))
    ang = 2.0 * np.pi * z[:, 1]
    d = np.stack([sz * np.cos(ang), sz * np.sin(ang), cz], axis=1)
    s = (np.arange(n_beads, dtype=np.float64) - 0.5 * (n_beads - 1)) * bond
    X = c[:, None, :] + s[None, :, None] * d[:, None, :]
    return X.reshape(n, 3).astype(np.float32)


def lattice_cloud(nx, ny, nz, spacing, jitter=0.0, seed=0):
    """Primitive cubic lattice, optionally perturbed (the paper's accuracy clouds, L281)."""
    g = np.stack(np.meshgrid(np.arange(nx), np.arange(ny), np.arange(nz), indexing="ij"), -1)
    X = g.reshape(-1, 3).astype(np.float64) * spacing
    if jitter:
        X = X + (uniform01(seed, 0, X.size).reshape(X.shape) - 0.5) * 2.0 * jitter
    return X.astype(np.float32)


def line_points(n):
    """x_i = (i + 1/2)/n on the x axis: the 1-D example of Fig. 4."""
    X = np.zeros((n, 3), dtype=np.float64)
    X[:, 0] = (np.arange(n) + 0.5) / n
    return X.astype(np.float32)


# -------------------------------------------------------------------------------- forces
def gaussian_forces(n, seed=2):
    return normal01(seed, 2, 3 * n).reshape(n, 3).astype(np.float32)


def gravity_forces(n):
    F = np.zeros((n, 3), dtype=np.float32)
    F[:, 2] = -1.0
    return F


def filament_forces(X, n_chains, n_beads, bond=2.2, k=100.0, kappa=10.0, xp=np):
    """Harmonic bonds (Eq. 12) + bending from kappa*(1 - t1.t2) (Eq. 13 with
    cos(theta) = -t1.t2) + gravity (0,0,-1).  Input generation only.  `xp` may be numpy
    or torch (same operators) so that multi-step runs can keep X on the device."""
    P = X.reshape(n_chains, n_beads, 3)
    F = xp.zeros_like(P)
    F[:, :, 2] -= 1.0
    r = P[:, 1:, :] - P[:, :-1, :]
    d = xp.sqrt((r * r).sum(-1))[..., None]
    t = r / d
    ft = k * (d - bond) * t                      # on bead i, opposite on i+1
    F[:, :-1, :] += ft
    F[:, 1:, :] -= ft
    if n_beads >= 3:
        t1, t2 = t[:, :-1, :], t[:, 1:, :]
        d1, d2 = d[:, :-1, :], d[:, 1:, :]
        c = (t1 * t2).sum(-1)[..., None]
        fm = -kappa * (t2 - c * t1) / d1         # bead i-1
        fp = kappa * (t1 - c * t2) / d2          # bead i+1
        F[:, :-2, :] += fm
        F[:, 2:, :] += fp
        F[:, 1:-1, :] -= fm + fp
    return F.reshape(-1, 3)


# --------------------------------------------------------------------------- MLP weights
def xavier_mlp(dims, seed, bias_scale=0.0):
    """Xavier-uniform weights, gain 1, drawn layer by layer (stream = layer index), row-major
    W[l] of shape [out][in]; biases zero unless bias_scale > 0 (tests cover non-zero biases).
    Returns (Ws, bs) as lists of float32 arrays."""
    Ws, bs = [], []
    for l in range(len(dims) - 1):
        fi, fo = dims[l], dims[l + 1]
        bound = math.sqrt(6.0 / (fi + fo))
        W = (uniform01(seed, 10 + l, fi * fo) * 2.0 - 1.0) * bound
        Ws.append(W.reshape(fo, fi).astype(np.float32))
        if bias_scale > 0.0:
            b = (uniform01(seed, 50 + l, fo) * 2.0 - 1.0) * bias_scale
        else:
            b = np.zeros(fo)
        bs.append(b.astype(np.float32))
    return Ws, bs


# ------------------------------------------------------------------------------- configs
CONFIGS = {
    # name: BASELINE.json config it realises
    "c1": dict(n=2048, shape="cube", phi=0.1, forces="gaussian", leaf=64, eta=1.0, tol=1e-4,
               rcut3=0.0, steps=1, dt=0.0),
    "c2": dict(n=65536, shape="ball", phi=0.2, forces="gravity", leaf=64, eta=1.0, tol=1e-4,
               rcut3=4.0, steps=10, dt=0.01),
    "c3": dict(n=1048576, shape="cube", phi=0.1, forces="gaussian", leaf=64, eta=1.0, tol=1e-4,
               rcut3=4.0, steps=1, dt=0.0),
    "c4": dict(n=10000000, shape="cube", phi=0.05, forces="gaussian", leaf=128, eta=1.0, tol=1e-4,
               rcut3=4.0, steps=1, dt=0.0),
    "c5": dict(n=1000000, shape="chains", phi=0.1, forces="filament", leaf=64, eta=1.0, tol=1e-4,
               rcut3=4.0, steps=100, dt=0.005, n_chains=20000, n_beads=50, kappa_max=50.0),   # S-18b: chains need 50 for the 1e-5 bar
}


def config(name, n=None):
    """(cfg dict, X, F) for a named config; `n` overrides the particle count while keeping
    the volume fraction (used for bounded CPU samples of the same workload)."""
    cfg = dict(CONFIGS[name])
    if n is not None:
        if cfg["shape"] == "chains":
            cfg["n_chains"] = max(1, n // cfg["n_beads"])
            n = cfg["n_chains"] * cfg["n_beads"]
        cfg["n"] = n
    n = cfg["n"]
    if cfg["shape"] == "cube":
        X = cube_cloud(n, cfg["phi"], seed=0)
    elif cfg["shape"] == "ball":
        X = ball_cloud(n, cfg["phi"], seed=0)
    else:
        X = chain_cloud(cfg["n_chains"], cfg["n_beads"], cfg["phi"], seed=0)
    if cfg["forces"] == "gaussian":
        F = gaussian_forces(n, seed=2)
    elif cfg["forces"] == "gravity":
        F = gravity_forces(n)
    else:
        F = filament_forces(X.astype(np.float64), cfg["n_chains"], cfg["n_beads"]).astype(np.float32)
    return cfg, X, F
