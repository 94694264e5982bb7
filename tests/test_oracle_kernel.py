"""Pins for the oracle's MLP, two-body entry, dense product, three-body term and Euler step.

Each pin is a closed form, an invariant or a special case fixed by the paper / the mathematics
(SURVEY 8(c) "What pins each part"), chosen so that a dropped term, wrong sign/index or a
transposed operand fails at least one of them.  Nothing here re-types the oracle's formula.
"""
import math
import numpy as np
import pytest
import oracle
import synth
from conftest import zero_mlp, rel_l2

D2 = synth.MLP2_DIMS
D3 = synth.MLP3_DIMS
EYE = np.eye(3).ravel()


def one_hot_chain(dims, i_in, h1, h2, o, w1, w2, w3, b=(0.0, 0.0, 0.0)):
    """MLP whose only non-zero path is in[i_in] -> hidden1[h1] -> hidden2[h2] -> out[o]."""
    Ws, bs = zero_mlp(dims)
    Ws[0][h1, i_in] = w1
    Ws[1][h2, h1] = w2
    Ws[2][o, h2] = w3
    bs[0][h1], bs[1][h2], bs[2][o] = b
    return Ws, bs


# ------------------------------------------------------------------ MLP orientation / activation
def test_mlp_one_hot_chain_closed_form():
    # y[o] = w3 tanh(w2 tanh(w1 x[i] + b1) + b2) + b3 ; W[l] is [out][in]; no tanh on the output (S-4)
    x = np.array([0.3, -0.7, 0.2, 1.9])
    m = one_hot_chain(D2, 2, 5, 9, 4, 0.7, 1.3, -2.5, b=(0.1, -0.2, 3.0))
    y = oracle.mlp_forward(m, x)
    want = -2.5 * math.tanh(1.3 * math.tanh(0.7 * 0.2 + 0.1) - 0.2) + 3.0
    assert abs(y[4] - want) < 1e-6 * abs(want)          # weights are stored as fp32
    assert np.all(np.delete(y, 4) == 0.0)
    assert abs(y[4]) > 1.0                                # no activation on the last layer


def test_mlp_zero_weights_gives_last_bias():
    m = zero_mlp(D2, b_last=np.arange(9) + 1.0)
    assert np.allclose(oracle.mlp_forward(m, np.ones(4)), np.arange(9) + 1.0)


# --------------------------------------------------------------------------- two-body entry
def test_entry_zero_weights_is_bias_over_r():
    b3 = np.arange(9) * 0.5 - 1.0
    m = zero_mlp(D2, b_last=b3)
    M = oracle.entry2(m, 1.0, [1, 2, 3], [4, 6, 3])      # r = (3,4,0), |r| = 5
    assert np.allclose(M, b3.reshape(3, 3) / 5.0, rtol=1e-12)   # S-3 row-major, Eq. (4) 1/r


def test_entry_direction_features_and_a_over_r():
    # S-1: r_ij = X_j - X_i ; S-2 features [r_hat, a/r]
    Xi, Xj = [0, 0, 0], [2, 0, 0]
    m = one_hot_chain(D2, 0, 1, 2, 0, 1.0, 1.0, 1.0)
    v = math.tanh(math.tanh(1.0)) / 2.0
    assert abs(oracle.entry2(m, 1.0, Xi, Xj)[0, 0] - v) < 1e-12
    assert abs(oracle.entry2(m, 1.0, Xj, Xi)[0, 0] + v) < 1e-12          # swapping flips r_hat
    m = one_hot_chain(D2, 1, 1, 2, 5, 1.0, 1.0, 1.0)                      # y component -> out[5] = R[1][2]
    M = oracle.entry2(m, 1.0, [0, 0, 0], [0, -4, 0])
    assert abs(M[1, 2] + math.tanh(math.tanh(1.0)) / 4.0) < 1e-12 and M[2, 1] == 0
    m = one_hot_chain(D2, 3, 0, 0, 8, 1.0, 1.0, 1.0)                      # a/r feature
    M = oracle.entry2(m, 2.0, [0, 0, 0], [0, 0, 4])
    assert abs(M[2, 2] - math.tanh(math.tanh(0.5)) / 4.0) < 1e-12


def test_entry_homogeneity(mlp2):
    # zero biases: scaling X and a by s keeps the features, so M scales by 1/s (SURVEY pins)
    Xi, Xj = np.array([1.0, 2.0, -1.0]), np.array([4.0, -2.0, 3.0])
    M1 = oracle.entry2(mlp2, 1.0, Xi, Xj)
    M4 = oracle.entry2(mlp2, 4.0, 4 * Xi, 4 * Xj)       # powers of two: exact in fp32
    assert np.allclose(M4, M1 / 4.0, rtol=1e-13)
    assert np.abs(M1).max() > 1e-3


def test_coincident_centres_stay_finite(mlp2_bias):
    M = oracle.entry2(mlp2_bias, 1.0, [1, 1, 1], [1, 1, 1])              # S-7 clamp
    assert np.all(np.isfinite(M))


# ----------------------------------------------------------------------------- dense product
def test_dense_identity_kernel_is_coulomb_sum():
    # weights 0, b3 = vec(I): M_ij = I/r, so U - F is three independent Coulomb-type sums
    m = zero_mlp(D2, b_last=EYE)
    X = synth.cube_cloud(60, 0.1, seed=5)
    F = synth.gaussian_forces(60, seed=6)
    U = oracle.dense_matvec(X, F, m)
    Xd = X.astype(np.float64)
    D = np.linalg.norm(Xd[:, None] - Xd[None], axis=-1)
    np.fill_diagonal(D, np.inf)
    want = F.astype(np.float64) + (1.0 / D) @ F.astype(np.float64)
    assert rel_l2(U, want) < 1e-13                       # includes S-5: self term F_i, no j = i
    U0 = oracle.dense_matvec(X, F, m, include_self=False)
    assert rel_l2(U0, want - F) < 1e-13


def test_dense_row_major_block_action():
    # R[0][1] = 1 only: U_i[0] = F_i[0] + sum_j F_j[1]/r_ij ; other components untouched (S-3)
    b3 = np.zeros(9)
    b3[1] = 1.0
    m = zero_mlp(D2, b_last=b3)
    X = synth.cube_cloud(20, 0.1, seed=7)
    F = synth.gaussian_forces(20, seed=8)
    U = oracle.dense_matvec(X, F, m)
    Xd = X.astype(np.float64)
    D = np.linalg.norm(Xd[:, None] - Xd[None], axis=-1)
    np.fill_diagonal(D, np.inf)
    assert np.allclose(U[:, 0], F[:, 0] + (1.0 / D) @ F[:, 1].astype(np.float64), rtol=1e-12)
    assert np.allclose(U[:, 1:], F[:, 1:], rtol=0, atol=0)


def test_dense_invariants(mlp2_bias):
    n = 80
    X = np.round(synth.cube_cloud(n, 0.1, seed=9) * 64) / 64          # dyadic: translations are exact
    F = synth.gaussian_forces(n, seed=10)
    G = synth.gaussian_forces(n, seed=11)
    U = oracle.dense_matvec(X, F, mlp2_bias)
    # translation invariance (HIs depend only on relative positions)
    Ut = oracle.dense_matvec((X + np.float32([8.0, -16.0, 4.0])).astype(np.float32), F, mlp2_bias)
    assert rel_l2(Ut, U) < 1e-13
    # linearity in F
    Ug = oracle.dense_matvec(X, G, mlp2_bias)
    Us = oracle.dense_matvec(X, (2 * F + 0.5 * G).astype(np.float32), mlp2_bias)
    assert rel_l2(Us, 2 * U + 0.5 * Ug) < 1e-6           # 2F + G/2 is re-rounded to fp32
    # permutation equivariance
    p = np.random.default_rng(0).permutation(n)
    Up = oracle.dense_matvec(X[p], F[p], mlp2_bias)
    assert rel_l2(Up, U[p]) < 1e-13
    # rows subset agrees with the full product
    rows = np.array([3, 17, 42])
    assert np.allclose(oracle.dense_matvec(X, F, mlp2_bias, rows=rows), U[rows], rtol=1e-14)
    # no symmetry is assumed (S-1): M_ij != M_ji^T for a random MLP
    Mij = oracle.entry2(mlp2_bias, 1.0, X[0], X[1])
    Mji = oracle.entry2(mlp2_bias, 1.0, X[1], X[0])
    assert not np.allclose(Mij, Mji.T)


# -------------------------------------------------------------------------------- three-body
def clustered(n, seed, side):
    return (synth.uniform01(seed, 0, 3 * n).reshape(n, 3) * side).astype(np.float32)


def test_three_body_hand_case():
    # weights 0, b3 = vec(I): face (j,k,i) adds F_j / (|X_j-X_k| |X_k-X_i|) (Eq. (4), S-23)
    m = zero_mlp(D3, b_last=EYE)
    X = np.float32([[0, 0, 0], [3, 0, 0], [0, 2, 0]])
    F = np.float32([[1, 0, 0], [0, 1, 0], [0, 0, 1]])
    U, nf = oracle.three_body(X, F, m, 4.0, brute=True)
    d = lambda p, q: np.linalg.norm(X[p].astype(np.float64) - X[q])
    want = np.zeros((3, 3))
    for i in range(3):
        for j in range(3):
            for k in range(3):
                if len({i, j, k}) == 3 and d(i, k) < 4 and d(j, k) < 4:
                    want[i] += F[j] / (d(j, k) * d(k, i))
    assert nf == 6 and np.allclose(U, want, rtol=1e-13)
    # |X_1 - X_2| = sqrt(13) < 4, so all six faces exist; shrink the cutoff to 3.5: N(0) = {1,2},
    # N(1) = {0}, N(2) = {0} -> only faces with k = 0 remain: (1,0,2) and (2,0,1)
    U2, nf2 = oracle.three_body(X, F, m, 3.5, brute=True)
    assert nf2 == 2
    assert np.allclose(U2[2], F[1] / (3.0 * 2.0)) and np.allclose(U2[1], F[2] / (2.0 * 3.0)) and np.all(U2[0] == 0)


def test_three_body_feature_order():
    X = np.float32([[0, 0, 0], [1, 2, 0.5], [-1, 0.5, 1]])      # i = 0, j = 1, k = 2 and all perms
    F = np.float32([[1, 0, 0], [1, 0, 0], [1, 0, 0]])
    Xd = X.astype(np.float64)
    for idx in range(7):
        m = one_hot_chain(D3, idx, 3, 4, 0, 0.5, 1.0, 1.0)
        U, nf = oracle.three_body(X, F, m, 10.0, brute=True)
        assert nf == 6
        want = 0.0
        i = 0
        for j, k in ((1, 2), (2, 1)):
            feat = np.concatenate([Xd[j] - Xd[i], Xd[k] - Xd[i], [np.linalg.norm(Xd[j] - Xd[k])]])
            want += math.tanh(math.tanh(0.5 * feat[idx])) / (np.linalg.norm(Xd[j] - Xd[k]) * np.linalg.norm(Xd[k] - Xd[i]))
        assert abs(U[0, 0] - want) < 1e-12, idx


def test_three_body_cell_list_equals_triple_loop_and_face_count(mlp3):
    n = 150
    X = clustered(n, 21, 14.0)
    F = synth.gaussian_forces(n, seed=22)
    Ub, nfb = oracle.three_body(X, F, mlp3, 4.0, brute=True)
    Uc, nfc = oracle.three_body(X, F, mlp3, 4.0, brute=False)
    assert nfb == nfc and nfb > 1000
    assert rel_l2(Uc, Ub) < 1e-12
    # N_f = sum_k d_k (d_k - 1) (L74), degrees from the fp32 distance rule
    dx = X[:, None, :] - X[None, :, :]
    d2 = (dx[..., 0] * dx[..., 0] + dx[..., 1] * dx[..., 1]) + dx[..., 2] * dx[..., 2]
    deg = (d2 < np.float32(16.0)).sum(1) - 1
    assert nfb == int((deg * (deg - 1)).sum())


def test_three_body_cutoff_is_strict(mlp3):
    F = np.float32([[1, 0, 0]] * 3)
    X = np.float32([[0, 0, 0], [4, 0, 0], [0, 4, 0]])         # both neighbours at exactly Rcut
    assert oracle.three_body(X, F, mlp3, 4.0)[1] == 0 and oracle.three_body(X, F, mlp3, 4.0, brute=True)[1] == 0
    X[1, 0] = X[2, 1] = np.float32(3.999)
    assert oracle.three_body(X, F, mlp3, 4.0)[1] == 2          # faces (1,0,2) and (2,0,1) only
    assert oracle.three_body(X, F, mlp3, 0.0)[1] == 0


# -------------------------------------------------------------------------------------- step
def test_euler_step_by_hand():
    X = np.float32([[1, 2, 3], [4, 5, 6]])
    U = np.array([[0.5, -1.0, 2.0], [0.0, 0.0, -4.0]])
    Y = oracle.euler(X, U, 0.25)
    assert np.array_equal(Y, np.float32([[1.125, 1.75, 3.5], [4, 5, 5]]))
    assert np.array_equal(oracle.euler(X, np.zeros((2, 3)), 0.25), X)


def test_zero_force_means_zero_velocity(mlp2_bias, mlp3):
    X = synth.cube_cloud(40, 0.1, seed=3)
    F = np.zeros((40, 3), np.float32)
    assert np.all(oracle.dense_matvec(X, F, mlp2_bias) == 0)
    assert np.all(oracle.three_body(X, F, mlp3, 4.0)[0] == 0)


# ---- self terms M^(s,2), M^(s,3) of Eq. (6) (Eq. (2)): 18-output networks [alpha^(s), alpha^(t)] ----
def _np_mlp(mlp, x):
    """numpy restatement of y = W_L tanh(... tanh(W_1 x + b_1) ...) + b_L, independent of the oracle's code"""
    Ws, bs = mlp
    h = np.asarray(x, np.float64)
    for l, (W, b) in enumerate(zip(Ws, bs)):
        h = W.astype(np.float64) @ h + b.astype(np.float64)
        if l + 1 < len(Ws):
            h = np.tanh(h)
    return h


def test_self_terms_against_numpy_brute_force():
    import synth
    n, rcut = 36, 4.0
    X = synth.cube_cloud(n, 0.15, seed=8)
    F = synth.gaussian_forces(n, seed=9)
    m2 = synth.xavier_mlp((4, 32, 32, 18), 1, bias_scale=0.2)
    m3 = synth.xavier_mlp((7, 64, 64, 18), 3, bias_scale=0.2)
    U, npairs, nf = oracle.self_terms(X, F, m2, m3, rcut)
    Xd, Fd = X.astype(np.float64), F.astype(np.float64)
    inside = lambda p, q: np.float32(((X[p] - X[q]) ** 2).sum()) < np.float32(rcut * rcut)
    ref = np.zeros((n, 3))
    cnt2 = cnt3 = 0
    for i in range(n):
        for j in range(n):
            if j == i or not inside(j, i):
                continue
            r = Xd[j] - Xd[i]
            d = np.linalg.norm(r)
            y = _np_mlp(m2, [r[0] / d, r[1] / d, r[2] / d, 1.0 / d])
            ref[i] += (y[:9].reshape(3, 3) / d) @ Fd[i]                    # alpha_2^(s) acts on F_i
            cnt2 += 1
    for k in range(n):
        nb = [p for p in range(n) if p != k and inside(p, k)]
        for i in nb:
            for j in nb:
                if i == j:
                    continue
                djk, dki = np.linalg.norm(Xd[j] - Xd[k]), np.linalg.norm(Xd[k] - Xd[i])
                y = _np_mlp(m3, np.concatenate([Xd[j] - Xd[i], Xd[k] - Xd[i], [djk]]))
                ref[i] += (y[:9].reshape(3, 3) / (djk * dki)) @ Fd[i]        # alpha_3^(s) acts on F_i
                cnt3 += 1
    assert (npairs, nf) == (cnt2, cnt3) and cnt2 > 0 and cnt3 > 0
    assert rel_l2(U, ref) < 1e-12


def test_self_terms_special_cases():
    import synth
    n, rcut = 60, 5.0
    X = synth.cube_cloud(n, 0.1, seed=2)
    F = synth.gaussian_forces(n, seed=3)
    # 9-output networks have no self half: nothing is added
    U0, p0, f0 = oracle.self_terms(X, F, synth.xavier_mlp((4, 32, 32, 9), 1), synth.xavier_mlp((7, 64, 64, 9), 3), rcut)
    assert np.all(U0 == 0) and (p0, f0) == (0, 0)
    # all weights zero, b_last = [vec(I), anything]: alpha_2^(s) = I / r, so U_i = F_i * sum_{j in N(i)} 1 / r_ij (closed form)
    Ws, bs = zero_mlp((4, 32, 32, 18), b_last=np.concatenate([np.eye(3).ravel(), np.full(9, 7.0)]))
    U1, p1, _ = oracle.self_terms(X, F, (Ws, bs), None, rcut)
    D = np.linalg.norm(X[:, None, :].astype(np.float64) - X[None, :, :].astype(np.float64), axis=-1)
    inside = (((X[:, None, :] - X[None, :, :]) ** 2).sum(-1).astype(np.float32) < np.float32(rcut * rcut)) & ~np.eye(n, dtype=bool)
    s = np.where(inside, 1.0 / np.where(D > 0, D, 1.0), 0.0).sum(1)
    assert p1 == int(inside.sum()) and rel_l2(U1, F.astype(np.float64) * s[:, None]) < 1e-13
    # the transverse half of an 18-output network is what the H-matrix entry and the three-body term use: with the halves swapped
    # in the last layer the entry of one network is the self entry of the other
    m2 = synth.xavier_mlp((4, 32, 32, 18), 1, bias_scale=0.1)
    Wsw = [w.copy() for w in m2[0]]; bsw = [b.copy() for b in m2[1]]
    Wsw[-1] = np.concatenate([m2[0][-1][9:], m2[0][-1][:9]]); bsw[-1] = np.concatenate([m2[1][-1][9:], m2[1][-1][:9]])
    m9 = (m2[0][:-1] + [m2[0][-1][9:]], m2[1][:-1] + [m2[1][-1][9:]])
    assert np.array_equal(oracle.entry2(m2, 1.0, X[0], X[1]), oracle.entry2(m9, 1.0, X[0], X[1]))
    Ua, _, _ = oracle.self_terms(X, F, (Wsw, bsw), None, rcut)
    ref = np.zeros((n, 3))
    for i in range(n):
        for j in np.flatnonzero(inside[i]):
            ref[i] += oracle.entry2(m9, 1.0, X[i], X[j]) @ F[i].astype(np.float64)
    assert rel_l2(Ua, ref) < 1e-13
    # three-body: the transverse half of an 18-output network equals the 9-output network made of that half
    m3 = synth.xavier_mlp((7, 64, 64, 18), 3, bias_scale=0.1)
    m3t = (m3[0][:-1] + [m3[0][-1][9:]], m3[1][:-1] + [m3[1][-1][9:]])
    Ut, nft = oracle.three_body(X, F, m3, rcut)
    Ut9, nf9 = oracle.three_body(X, F, m3t, rcut)
    assert nft == nf9 and np.array_equal(Ut, Ut9)
