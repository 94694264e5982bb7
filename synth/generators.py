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
MLP2_PAPER_DIMS = (4, 128, 512, 128, 9)   # the paper's hidden layers 128 / 512 / 128 on the configs' features / outputs


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


def lattice_drop(radius, phi, centre=(0.0, 0.0, 0.0), jitter=0.2, seed=0, a=1.0):
    """One suspension drop as the paper builds it (Sec. 4.3.1): a primitive cubic lattice at volume
    fraction phi (spacing h = a (4 pi / 3 / phi)^(1/3)), the points outside the sphere discarded, every position
    slightly perturbed (uniform in +-jitter per axis; non-overlapping while h - 2 sqrt(3) jitter > 2a).  The sphere
    centre sits on a lattice point.  The number of particles follows from the lattice; the paper's drop of radius 175
    at phi = 10 % has 523,305 (its lattice offset is not stated; this one has 536,393)."""
    h = a * (4.0 * math.pi / 3.0 / phi) ** (1.0 / 3.0)
    k = int(math.floor(radius / h)) + 1
    ax = np.arange(-k, k + 1, dtype=np.float64) * h
    g = np.stack(np.meshgrid(ax, ax, ax, indexing="ij"), -1).reshape(-1, 3)
    g = g[(g * g).sum(1) <= radius * radius]
    if jitter:
        g = g + (uniform01(seed, 0, g.size).reshape(g.shape) - 0.5) * 2.0 * jitter
    return (g + np.asarray(centre, np.float64)).astype(np.float32)


def two_drops(radius=175.0, phi=0.1, gap=0.2, jitter=0.2, seed=0):
    """The two sedimenting drops of PAPER.md L342: vertically aligned, no horizontal offset, the trailing drop above the
    leading one.  The initial separation is not stated in the text; `gap` (in radii) is the clearance between the spheres."""
    lead = lattice_drop(radius, phi, (0.0, 0.0, 0.0), jitter, seed)
    trail = lattice_drop(radius, phi, (0.0, 0.0, (2.0 + gap) * radius), jitter, seed + 1)
    return np.concatenate([lead, trail], 0)


def filament_sphere(n_fil=5120, n_beads=21, r_b=3.0, n_free=107520, dmin=2.1, seed=0, a=1.0):
    """The mixture of PAPER.md L369 (Sec. 4.3.2): n_fil straight filaments of n_beads beads (spacing r_b), randomly
    oriented and positioned inside the inner sphere R_in = 2^(-1/3) R_out, R_out = 4 * 10^(1/3) (n_beads - 1) r_b, and n_free
    individual particles in the shell between R_in and R_out; any two beads / particles of different objects at least
    dmin apart.  Random sequential addition in counter order: a candidate that comes within dmin of an earlier
    object is dropped.  Filaments come first in the output (n_fil * n_beads rows), then the free particles.
    "Positioned within the inner sphere" is read as: every bead inside it."""
    from scipy.spatial import cKDTree
    R_out = 4.0 * 10.0 ** (1.0 / 3.0) * (n_beads - 1) * r_b
    R_in = 0.5 ** (1.0 / 3.0) * R_out
    half = 0.5 * (n_beads - 1) * r_b
    s = (np.arange(n_beads, dtype=np.float64) - 0.5 * (n_beads - 1)) * r_b

    def sphere_dirs(u):
        cz = 2.0 * u[:, 0] - 1.0
        sz = np.sqrt(np.maximum(0.0, 1.0 - cz * cz))
        ang = 2.0 * np.pi * u[:, 1]
        return np.stack([sz * np.cos(ang), sz * np.sin(ang), cz], 1)

    def add_batch(have, cand):
        """cand [n_obj][n_pts][3] in counter order: drop objects within dmin of `have` [*][3] or of an EARLIER kept candidate"""
        n_obj, n_pts = cand.shape[:2]
        keep = np.ones(n_obj, bool)
        pts = cand.reshape(-1, 3)
        if len(have):
            hit = np.isfinite(cKDTree(have).query(pts, k=1, distance_upper_bound=dmin)[0])
            keep &= ~hit.reshape(n_obj, n_pts).any(1)
        pairs = cKDTree(pts).query_pairs(dmin, output_type="ndarray")
        if len(pairs):
            oi, oj = pairs[:, 0] // n_pts, pairs[:, 1] // n_pts
            sel = oi != oj
            lo, hi = np.minimum(oi[sel], oj[sel]), np.maximum(oi[sel], oj[sel])
            order = np.lexsort((hi, lo))
            for i, j in zip(lo[order], hi[order]):
                if keep[i]:
                    keep[j] = False                                  # the later object of a close pair goes
        return cand[keep]

    # filaments: centre uniform in the ball (rejection from the cube), kept if both end beads are inside the inner sphere
    fil = np.zeros((0, n_beads, 3))
    start = 0
    while len(fil) < n_fil:
        m = int((n_fil - len(fil)) * 3.0) + 64
        c = (uniform01(seed, 0, 3 * m, start=3 * start).reshape(m, 3) * 2.0 - 1.0) * R_in
        d = sphere_dirs(uniform01(seed, 4, 2 * m, start=2 * start).reshape(m, 2))
        start += m
        ends_ok = (np.linalg.norm(c + half * d, axis=1) <= R_in - a) & (np.linalg.norm(c - half * d, axis=1) <= R_in - a)
        cand = (c[:, None, :] + s[None, :, None] * d[:, None, :])[ends_ok]
        fil = np.concatenate([fil, add_batch(fil.reshape(-1, 3), cand)], 0)[:n_fil]
    beads = fil.reshape(-1, 3)
    # free particles in the shell, against the filaments and against each other
    free = np.zeros((0, 3))
    start = 0
    while len(free) < n_free:
        m = int((n_free - len(free)) * 2.6) + 256
        c = (uniform01(seed, 6, 3 * m, start=3 * start).reshape(m, 3) * 2.0 - 1.0) * R_out
        start += m
        r = np.linalg.norm(c, axis=1)
        c = c[(r >= R_in + a) & (r <= R_out - a)]
        if len(c):
            free = np.concatenate([free, add_batch(np.concatenate([beads, free], 0), c[:, None, :])[:, 0, :]], 0)[:n_free]
    return np.concatenate([beads, free], 0).astype(np.float32), dict(R_out=R_out, R_in=R_in, L_f=(n_beads - 1) * r_b + 2 * a)


def mixture_forces(X, n_fil, n_beads, bond=3.0, k=20.0, kappa=50.0, xp=np):
    """Forces of the filament mixture: harmonic tension k_t = 20 with rest length r_b, COS bending
    k_b = 50 on the filament beads (the first n_fil * n_beads rows), gravity (0,0,-1) on every particle."""
    nf = n_fil * n_beads
    F = xp.zeros_like(X)
    F[:, 2] -= 1.0
    Ff = filament_forces(X[:nf], n_fil, n_beads, bond=bond, k=k, kappa=kappa, xp=xp)
    Ff[:, 2] += 1.0                                                  # filament_forces adds gravity itself
    F[:nf] += Ff
    return F


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
# kappa_max: 0 = Alg. 2 as printed (the default of the library and of the oracle); c5 opts in to S-18b.
# near_path: 2 = near-field entries on the tcgen05 tensor cores with split tf32 operands (fp32-class accuracy).
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
    # the paper's own workloads at the paper's parameters; random-init MLPs
    "p1": dict(n=None, shape="two_drops", phi=0.1, forces="gravity", leaf=50, eta=1.0, tol=0.1, rcut3=4.0, steps=50, dt=0.01,
               radius=175.0),
    "p2": dict(n=215040, shape="filament_sphere", phi=None, forces="mixture", leaf=50, eta=1.0, tol=0.02, rcut3=4.0, steps=1,
               dt=0.002, n_chains=5120, n_beads=21, n_free=107520),
}


def config(name, n=None):
    """(cfg dict, X, F) for a named config; `n` overrides the particle count while keeping
    the volume fraction (used for bounded CPU samples of the same workload)."""
    cfg = dict(CONFIGS[name])
    if cfg["shape"] == "two_drops":
        scale = 1.0 if n is None else (n / 1072786.0) ** (1.0 / 3.0)      # n shrinks the radius at the same volume fraction
        X = two_drops(cfg["radius"] * scale, cfg["phi"])
        cfg["n"] = len(X)
        return cfg, X, gravity_forces(len(X))
    if cfg["shape"] == "filament_sphere":
        f = 1.0 if n is None else n / cfg["n"]
        cfg["n_chains"], cfg["n_free"] = max(1, int(cfg["n_chains"] * f)), max(1, int(cfg["n_free"] * f))
        X, _ = filament_sphere(cfg["n_chains"], cfg["n_beads"], 3.0, cfg["n_free"])
        cfg["n"] = len(X)
        F = mixture_forces(X.astype(np.float64), cfg["n_chains"], cfg["n_beads"]).astype(np.float32)
        return cfg, X, F
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
