"""Input generators: determinism, shapes, the closed forms the paper prints for its workloads."""
import math
import numpy as np
import synth


def test_rng_streams_are_counter_based():
    a = synth.uniform01(7, 3, 100)
    b = synth.uniform01(7, 3, 50, start=50)
    assert np.array_equal(a[50:], b)                       # counter based: a suffix can be drawn alone
    assert not np.array_equal(a, synth.uniform01(7, 4, 100))
    assert not np.array_equal(a, synth.uniform01(8, 3, 100))
    assert a.min() >= 0.0 and a.max() < 1.0
    assert np.array_equal(a.astype(np.float32).astype(np.float64), a)   # 24-bit: exact in fp32


def test_normal_moments():
    z = synth.normal01(2, 2, 200000)
    assert abs(z.mean()) < 0.01 and abs(z.std() - 1.0) < 0.01
    assert abs((z ** 3).mean()) < 0.03 and abs((z ** 4).mean() - 3.0) < 0.08


def test_cube_cloud_volume_fraction():
    n, phi = 2048, 0.1
    X = synth.cube_cloud(n, phi)
    L = synth.generators.cube_side(n, phi)
    assert abs(L - 44.1) < 0.05                            # C1 side 44.1
    assert X.dtype == np.float32 and X.shape == (n, 3)
    assert X.min() >= 0 and X.max() < L
    assert abs(n * 4 * math.pi / 3 / L ** 3 - phi) < 1e-12
    assert np.array_equal(X, synth.cube_cloud(n, phi))     # deterministic


def test_ball_cloud():
    n, phi = 4096, 0.2
    X = synth.ball_cloud(n, phi)
    R = (n / phi) ** (1 / 3)
    r = np.linalg.norm(X.astype(np.float64), axis=1)
    assert r.max() < R * (1 + 1e-6)
    assert abs((r < R / 2 ** (1 / 3)).mean() - 0.5) < 0.03    # uniform in volume
    # the accepted candidates come in counter order: a smaller drop is a scaled prefix
    R100 = (100 / phi) ** (1 / 3)
    assert np.allclose(synth.ball_cloud(100, phi) / R100, X[:100] / R, atol=1e-6)


def test_chain_cloud_geometry():
    X = synth.chain_cloud(50, 50, 0.1).astype(np.float64).reshape(50, 50, 3)
    bonds = np.linalg.norm(X[:, 1:] - X[:, :-1], axis=-1)
    assert np.allclose(bonds, 2.2, atol=1e-4)
    t = X[:, 1:] - X[:, :-1]
    t /= np.linalg.norm(t, axis=-1, keepdims=True)
    assert np.allclose((t[:, 1:] * t[:, :-1]).sum(-1), 1.0, atol=1e-5)   # straight


def test_filament_closed_forms_of_the_paper():
    # L_f = (N_b - 1) r_b + 2a = 62 for N_b = 21, r_b = 3; 5120 x 21 = 107,520
    assert (21 - 1) * 3 + 2 * 1 == 62
    assert 5120 * 21 == 107520 and 2 * 107520 == 215040
    R_out = 4 * 10 ** (1 / 3) * (21 - 1) * 3
    assert abs(0.5 ** (1 / 3) * R_out / R_out - 2 ** (-1 / 3)) < 1e-15


def test_filament_forces_are_minus_gradient_of_energy():
    nc, nb, bond, k, kappa = 3, 6, 2.2, 100.0, 10.0
    rng = np.random.default_rng(0)
    X = synth.chain_cloud(nc, nb, 0.1).astype(np.float64) + 0.2 * rng.standard_normal((nc * nb, 3))

    def energy(Y):
        P = Y.reshape(nc, nb, 3)
        r = P[:, 1:] - P[:, :-1]
        d = np.linalg.norm(r, axis=-1)
        t = r / d[..., None]
        e = 0.5 * k * ((d - bond) ** 2).sum()
        e += kappa * (1.0 - (t[:, 1:] * t[:, :-1]).sum(-1)).sum()
        e += P[:, :, 2].sum()                                  # gravity (0,0,-1)
        return e

    F = synth.filament_forces(X, nc, nb, bond, k, kappa)
    g = np.zeros_like(X)
    h = 1e-6
    for i in range(X.shape[0]):
        for c in range(3):
            Xp, Xm = X.copy(), X.copy()
            Xp[i, c] += h
            Xm[i, c] -= h
            g[i, c] = (energy(Xp) - energy(Xm)) / (2 * h)
    assert np.allclose(F, -g, atol=1e-5 * max(1.0, np.abs(g).max()))
    # internal forces sum to zero: net force is gravity only
    assert np.allclose(F.sum(0), [0, 0, -nc * nb], atol=1e-9)
    # straight chain at rest length: gravity only
    X0 = synth.chain_cloud(2, 5, 0.1).astype(np.float64)
    F0 = synth.filament_forces(X0, 2, 5, bond, k, kappa)
    assert np.allclose(F0, [[0, 0, -1]] * 10, atol=1e-3)


def test_xavier_bounds_and_shapes():
    Ws, bs = synth.xavier_mlp(synth.MLP2_DIMS, 1)
    assert [W.shape for W in Ws] == [(32, 4), (32, 32), (9, 32)]
    for W in Ws:
        bound = math.sqrt(6.0 / sum(W.shape))
        assert np.abs(W).max() <= bound and np.abs(W).max() > 0.8 * bound
    assert all(np.all(b == 0) for b in bs)
    _, bs2 = synth.xavier_mlp(synth.MLP2_DIMS, 1, bias_scale=0.3)
    assert all(np.abs(b).max() > 0 for b in bs2)


def test_configs_match_baseline_json():
    import json, os
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    txt = " ".join(json.load(open(os.path.join(root, "BASELINE.json")))["configs"])
    assert "N=2,048" in txt and synth.CONFIGS["c1"]["n"] == 2048
    assert "N=65,536" in txt and synth.CONFIGS["c2"]["n"] == 65536
    assert "N=1,048,576" in txt and synth.CONFIGS["c3"]["n"] == 1048576
    assert "N=10,000,000" in txt and synth.CONFIGS["c4"]["n"] == 10000000 and synth.CONFIGS["c4"]["leaf"] == 128
    assert "20,000 chains of 50 beads" in txt and synth.CONFIGS["c5"]["n_chains"] == 20000
    cfg, X, F = synth.config("c2", n=512)
    assert X.shape == (512, 3) and np.all(F == [0, 0, -1])


def test_two_drops_as_the_paper_builds_them():
    """lattice at phi = 10 %, points outside the sphere discarded, slightly perturbed; two drops vertically
    aligned.  At a reduced radius (the generator is the same at 175)."""
    R, phi = 40.0, 0.1
    X = synth.two_drops(R, phi).astype(np.float64)
    n1 = len(synth.lattice_drop(R, phi))
    assert len(X) == 2 * n1
    assert abs(n1 / (phi * R ** 3) - 1.0) < 0.03                     # N = phi R^3 / a^3 up to lattice discreteness
    lead, trail = X[:n1], X[n1:]
    assert np.abs(lead.mean(0)).max() < 0.2 and np.abs(trail.mean(0)[:2]).max() < 0.2      # no horizontal offset
    assert abs(trail.mean(0)[2] - 2.2 * R) < 0.2
    assert np.linalg.norm(lead, axis=1).max() <= R + 0.2 * math.sqrt(3) + 1e-4
    from scipy.spatial import cKDTree
    d, _ = cKDTree(X).query(X, k=2)
    h = (4 * math.pi / 3 / phi) ** (1 / 3)
    assert d[:, 1].min() >= h - 2 * 0.2 * math.sqrt(3) - 1e-4 > 2.0     # non-overlapping
    assert np.array_equal(synth.two_drops(R, phi), synth.two_drops(R, phi))


def test_filament_sphere_of_the_paper():
    """R_out = 4 * 10^(1/3) (N_b - 1) r_b, R_in = 2^(-1/3) R_out, filaments inside R_in, particles in the
    shell, minimum distance 2.1 between objects; equal numbers of filament beads and free particles."""
    nf, nb, nfree = 256, 21, 5376
    X, info = synth.filament_sphere(nf, nb, 3.0, nfree)
    X = X.astype(np.float64)
    assert len(X) == nf * nb + nfree and nf * nb == nfree
    assert abs(info["R_out"] - 4 * 10 ** (1 / 3) * 60) < 1e-9 and abs(info["R_in"] - info["R_out"] / 2 ** (1 / 3)) < 1e-9 and info["L_f"] == 62
    r = np.linalg.norm(X, axis=1)
    assert r[:nf * nb].max() <= info["R_in"] and r[nf * nb:].min() >= info["R_in"] and r.max() <= info["R_out"]
    P = X[:nf * nb].reshape(nf, nb, 3)
    assert np.allclose(np.linalg.norm(P[:, 1:] - P[:, :-1], axis=-1), 3.0, atol=1e-4)
    from scipy.spatial import cKDTree
    pairs = cKDTree(X).query_pairs(2.1 - 1e-4, output_type="ndarray")
    assert len(pairs) == 0
    F = synth.mixture_forces(X, nf, nb)
    assert np.allclose(F[nf * nb:], [0, 0, -1]) and np.abs(F[:nf * nb] - [0, 0, -1]).max() < 0.01    # straight, at rest length
    # a bent, stretched filament feels restoring forces that sum to zero (internal forces)
    Y = X.copy()
    Y[:nb] += np.random.default_rng(0).normal(0, 0.2, (nb, 3))
    G = synth.mixture_forces(Y, nf, nb)
    assert np.abs((G[:nb] - [0, 0, -1]).sum(0)).max() < 1e-9 and np.abs(G[:nb] - [0, 0, -1]).max() > 0.1
