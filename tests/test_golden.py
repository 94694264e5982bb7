"""Fixtures under tests/golden/: numbers the paper prints (L369) and the closed form of its 1-D example (Fig. 4)."""
import os

import numpy as np

import oracle
import synth

GOLD = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def read_kv(name):
    out = {}
    for line in open(os.path.join(GOLD, name)):
        if line.strip() and not line.startswith("#"):
            k, v = line.split()
            out[k] = float(v)
    return out


def test_filament_setup_numbers_of_the_paper():
    g = read_kv("paper_L369_filament_setup.txt")
    nb, rb = int(g["N_b"]), g["r_b"]
    assert (nb - 1) * rb + 2 * g["a"] == g["L_f"]                       # the paper's own formula and value
    assert g["n_filaments"] * nb == g["n_individual"] and g["n_individual"] * 2 == g["n_total"]
    # the chain generator builds exactly such filaments: straight, N_b beads, bond r_b -> end-to-end (N_b - 1) r_b
    X = synth.chain_cloud(7, nb, 0.05, bond=rb).reshape(7, nb, 3).astype(np.float64)
    ends = np.linalg.norm(X[:, -1] - X[:, 0], axis=1)
    assert np.allclose(ends + 2 * g["a"], g["L_f"], rtol=1e-5)
    bonds = np.linalg.norm(X[:, 1:] - X[:, :-1], axis=2)
    assert np.allclose(bonds, rb, rtol=1e-4)


def test_fig4_1d_partition_counts(mlp2):
    for line in open(os.path.join(GOLD, "fig4_1d_partition_counts.txt")):
        if not line.strip() or line.startswith("#"):
            continue
        f = [int(t) for t in line.split()]
        L, n_h, per_level = f[0], f[1], f[2:]
        n_leaf = 4
        H = oracle.HMatrix(synth.line_points(n_leaf * 2 ** L), mlp2, leaf=n_leaf, eta=1.0)
        assert H.nH == n_h
        lev = H.level[H.G[:, 0]]
        assert np.array_equal(lev, H.level[H.G[:, 1]])                   # equal leaves: blocks pair clusters of one level
        assert [int(np.sum(lev == l)) for l in range(2, L + 1)] == per_level
        assert int(np.sum(lev < 2)) == 0
