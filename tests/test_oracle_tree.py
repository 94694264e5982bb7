"""Pins for the oracle's Morton order, cluster tree (Def. 1), admissibility (Def. 2 / Eq. (7))
and BuildPartition (Alg. 1): brute force on tiny inputs, lattice closed forms, invariants and the
1-D example of Fig. 4."""
import numpy as np
import pytest
import oracle
import synth


def interleave_bruteforce(qx, qy, qz):
    """independent bit-by-bit Morton interleave with python ints (x highest in each triple)"""
    k = 0
    for b in range(21):
        k |= ((qx >> b) & 1) << (3 * b + 2)
        k |= ((qy >> b) & 1) << (3 * b + 1)
        k |= ((qz >> b) & 1) << (3 * b)
    return k


# ------------------------------------------------------------------------------------ Morton
def test_morton_keys_on_dyadic_lattice():
    # coordinates i/8, i = 0..8 -> ext = 1, q = i * 2^18 (and 2^21 - 1 at the far face) (S-8)
    g = np.arange(9) / 8.0
    X = np.stack(np.meshgrid(g, g, g, indexing="ij"), -1).reshape(-1, 3).astype(np.float32)
    keys = oracle.morton_keys(X)
    for p in range(0, len(X), 37):
        q = [min(int(round(v * 8)) << 18, (1 << 21) - 1) for v in X[p]]
        assert int(keys[p]) == interleave_bruteforce(*q)
    assert int(keys.max()) == (1 << 63) - 1 and int(keys.min()) == 0


def test_morton_bruteforce_random_and_axis_significance():
    X = synth.cube_cloud(200, 0.1, seed=12)
    keys = oracle.morton_keys(X)
    Xd = X.astype(np.float64)
    lo = Xd.min(0)
    ext = (Xd.max(0) - lo).max()                            # CUBE of the largest extent (S-8)
    for p in range(200):
        q = [min(int(np.floor((Xd[p, c] - lo[c]) / ext * 2097152.0)), 2097151) for c in range(3)]
        assert int(keys[p]) == interleave_bruteforce(*q)
    # x is the most significant axis of each triple (x is split first, Fig. 2)
    Y = np.float32([[0, 0, 0], [1, 1, 1], [0.5, 0, 0], [0.25, 0.99, 0.99]])
    k = oracle.morton_keys(Y)
    assert k[2] > k[3]


def test_morton_degenerate_extent():
    assert np.all(oracle.morton_keys(np.float32([[3, 4, 5]])) == 0)                 # N = 1
    assert np.all(oracle.morton_keys(np.float32([[3, 4, 5]] * 7)) == 0)             # all coincident


def test_order_is_stable_on_equal_keys(mlp2):
    # S-9: ascending key, ties by original index
    base = synth.cube_cloud(50, 0.1, seed=13)
    X = np.concatenate([base, base[::-1], base])            # every key occurs three times
    H = oracle.HMatrix(X, mlp2, leaf=4)
    k = oracle.morton_keys(X)
    assert np.array_equal(H.keys, k[H.perm])
    assert np.all(np.diff(H.keys.astype(np.float64)) >= 0)
    assert np.array_equal(H.perm, np.lexsort((np.arange(len(X)), k)))


# -------------------------------------------------------------------------------------- tree
def check_tree_invariants(H, leaf):
    n = H.n_nodes
    assert H.lo[0] == 0 and H.hi[0] == H.N and H.parent[0] == -1 and H.level[0] == 0
    internal = H.left >= 0
    assert np.all((H.right >= 0) == internal)
    cnt = H.hi - H.lo
    assert np.all(cnt[~internal] <= leaf) and np.all(cnt[internal] > leaf)           # S-10
    L, R = H.left[internal], H.right[internal]
    assert np.all(H.lo[L] == H.lo[internal]) and np.all(H.hi[R] == H.hi[internal])   # Def. 1(2)
    assert np.all(H.hi[L] == H.lo[R]) and np.all(H.hi[L] > H.lo[L]) and np.all(H.hi[R] > H.lo[R])
    assert np.all(R == L + 1)                                                          # BFS, left first
    assert np.all(H.parent[L] == np.nonzero(internal)[0]) and np.all(H.level[L] == H.level[internal] + 1)
    assert np.all(np.diff(H.level) >= 0)
    assert cnt[~internal].sum() == H.N and n == 2 * H.n_leaves - 1
    Xs = H.X[H.perm]
    for t in range(0, n, max(1, n // 200)):                                            # S-13 tight boxes
        assert np.array_equal(H.bmin[t], Xs[H.lo[t]:H.hi[t]].min(0))
        assert np.array_equal(H.bmax[t], Xs[H.lo[t]:H.hi[t]].max(0))


@pytest.mark.parametrize("leaf", [1, 7, 64])
def test_tree_invariants_random_cloud(mlp2, leaf):
    X = synth.cube_cloud(3000, 0.1, seed=14)
    H = oracle.HMatrix(X, mlp2, leaf=leaf)
    check_tree_invariants(H, leaf)
    # split rule S-11: the two sons differ in the highest differing key bit of the parent range
    for t in np.nonzero(H.left >= 0)[0][:300]:
        a, b = int(H.keys[H.lo[t]]), int(H.keys[H.hi[t] - 1])
        if a == b:
            continue
        bit = (a ^ b).bit_length() - 1
        m = H.hi[H.left[t]]
        assert (int(H.keys[m - 1]) >> bit) & 1 == 0 and (int(H.keys[m]) >> bit) & 1 == 1


def test_tree_on_dyadic_lattice_is_perfect(mlp2):
    X = synth.lattice_cloud(16, 16, 16, 1.0)                 # 4096 points, leaf 8 = 2x2x2 cells
    H = oracle.HMatrix(X, mlp2, leaf=8)
    check_tree_invariants(H, 8)
    assert H.n_leaves == 512 and H.n_nodes == 1023 and H.depth == 9
    leaves = H.left < 0
    assert np.all((H.hi - H.lo)[leaves] == 8)
    assert np.all((H.bmax - H.bmin)[leaves] == 1.0)          # each leaf is a 2x2x2 cell
    # alternating x, y, z bisection (Fig. 2): level-1 boxes split x, level-2 y, level-3 z
    for lvl, axis in ((1, 0), (2, 1), (3, 2)):
        ext = (H.bmax - H.bmin)[H.level == lvl]
        want = np.full(3, 15.0)
        want[:axis + 1] = 7.0
        assert np.all(ext == want)


def test_tree_equal_keys_split_at_median(mlp2):
    X = np.float32([[1, 1, 1]] * 10 + [[2, 2, 2]] * 3)
    H = oracle.HMatrix(X, mlp2, leaf=2)
    check_tree_invariants(H, 2)
    t = [i for i in range(H.n_nodes) if H.lo[i] == 0 and H.hi[i] == 10][0]
    assert H.hi[H.left[t]] == 5                               # lo + (hi - lo) / 2


def test_single_particle_and_tiny_inputs(mlp2):
    H = oracle.HMatrix(np.float32([[1, 2, 3]]), mlp2, leaf=64)
    assert H.n_nodes == 1 and H.nG == 0 and H.nH == 1
    H = oracle.HMatrix(synth.cube_cloud(5, 0.1), mlp2, leaf=64)
    assert H.n_nodes == 1 and H.nH == 1 and H.nG == 0


# ------------------------------------------------------------------- admissibility + Alg. 1
def numpy_admissible(H, t, s, eta):
    """Eq. (7) re-evaluated with numpy norms on the boxes (a hair of slack for rounding)."""
    if t == s:
        return False
    bt0, bt1 = H.bmin[t].astype(np.float64), H.bmax[t].astype(np.float64)
    bs0, bs1 = H.bmin[s].astype(np.float64), H.bmax[s].astype(np.float64)
    diam = max(np.linalg.norm(bt1 - bt0), np.linalg.norm(bs1 - bs0))
    gap = np.maximum(0.0, np.maximum(bt0 - bs1, bs0 - bt1))
    return diam <= eta * np.linalg.norm(gap) * (1 + 1e-12)


@pytest.mark.parametrize("n,leaf,eta,seed", [(1500, 16, 1.0, 15), (900, 8, 2.0, 16), (2048, 64, 1.0, 0), (700, 5, 0.5, 17)])
def test_partition_tiles_IxI_exactly_once(mlp2, n, leaf, eta, seed):
    X = synth.cube_cloud(n, 0.1, seed=seed)
    H = oracle.HMatrix(X, mlp2, leaf=leaf, eta=eta)
    cover = np.zeros((n, n), np.int16)
    for B in (H.G, H.H):
        for t, s in B:
            cover[H.lo[t]:H.hi[t], H.lo[s]:H.hi[s]] += 1
    assert cover.min() == 1 and cover.max() == 1
    leaves = H.left < 0
    assert np.all(leaves[H.H[:, 0]]) and np.all(leaves[H.H[:, 1]])                   # P^H is leaf x leaf
    for t, s in H.H[:: max(1, H.nH // 300)]:
        assert not H.admissible(t, s)
    for t, s in H.G[:: max(1, H.nG // 300)]:
        assert H.admissible(t, s) and numpy_admissible(H, t, s, eta)
        # maximality: the call of Alg. 1 that produced (t, s) was on an inadmissible pair.  Levels
        # stay equal until one side is a leaf, after which only the other side descends.
        if H.level[t] == H.level[s]:
            assert not H.admissible(H.parent[t], H.parent[s])
        elif H.level[t] > H.level[s]:
            assert H.left[s] < 0 and not H.admissible(H.parent[t], s)
        else:
            assert H.left[t] < 0 and not H.admissible(t, H.parent[s])
    # the partition is symmetric under (tau, sigma) <-> (sigma, tau)
    for name in "GH":
        T = H.block_table(name)
        Tt = T[:, [2, 3, 0, 1]]
        Tt = Tt[np.lexsort((Tt[:, 3], Tt[:, 2], Tt[:, 1], Tt[:, 0]))]
        assert np.array_equal(T, Tt)
    assert np.array_equal(H.admissible(1, 2), H.admissible(2, 1))


def test_diagonal_and_touching_boxes_never_admissible(mlp2):
    # S-15: a one-particle cluster has diam = dist = 0 against itself and must stay inadmissible
    X = np.float32([[0, 0, 0], [10, 0, 0]])
    H = oracle.HMatrix(X, mlp2, leaf=1, eta=1.0)
    assert H.n_nodes == 3 and H.nH == 2 and H.nG == 2        # (1,1),(2,2) near; (1,2),(2,1) far
    assert not H.admissible(1, 1) and H.admissible(1, 2)
    T = H.block_table("H")
    assert np.array_equal(T, [[0, 1, 0, 1], [1, 2, 1, 2]])


@pytest.mark.parametrize("L,n", [(4, 3), (6, 5), (8, 4)])
def test_fig4_one_dimensional_closed_form(mlp2, L, n):
    # Fig. 4 (L150, L188-L194): root [0,1], eta = 1.  With 2^L leaf intervals of n >= 3 points:
    # N^H = 3 * 2^L - 2 leaf blocks and 3 * 2^l - 6 admissible blocks at every level l >= 2.
    N = (1 << L) * n
    H = oracle.HMatrix(synth.line_points(N), mlp2, leaf=n, eta=1.0)
    assert H.n_leaves == 1 << L and H.depth == L and np.all((H.hi - H.lo)[H.left < 0] == n)
    assert H.nH == 3 * (1 << L) - 2
    lt, ls = H.level[H.G[:, 0]], H.level[H.G[:, 1]]
    assert np.array_equal(lt, ls)
    for lvl in range(0, L + 1):
        want = 3 * (1 << lvl) - 6 if lvl >= 2 else 0
        assert int((lt == lvl).sum()) == want
    # near blocks are exactly the index-distance <= 1 leaf pairs
    leaf_id = H.lo[H.H] // n
    assert np.all(np.abs(leaf_id[:, 0] - leaf_id[:, 1]) <= 1)


def test_eta_to_zero_leaves_only_single_particle_pairs_admissible(mlp2):
    X = synth.cube_cloud(600, 0.1, seed=18)
    H = oracle.HMatrix(X, mlp2, leaf=16, eta=1e-30)
    for t, s in H.G:
        assert H.hi[t] - H.lo[t] == 1 and H.hi[s] - H.lo[s] == 1       # S-15 consequence
    H2 = oracle.HMatrix(X, mlp2, leaf=16, eta=4.0)
    assert H2.nG > 0 and H2.nH < H.nH
