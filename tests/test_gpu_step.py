"""GPU parity: three-body graph term, self term / un-permute, Euler step."""
import numpy as np
import pytest

import oracle
import synth
from conftest import rel_l2
from gpu_util import f32, make_ctx, to_dev
from test_gpu_aca import gpu_replay

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("name,gen,forces", [
    ("ball", lambda: synth.ball_cloud(4000, 0.2), "gravity"),
    ("cube", lambda: synth.cube_cloud(3000, 0.1), "gauss"),
    ("chains", lambda: synth.chain_cloud(60, 50, 0.1), "gauss"),
    ("tiny", lambda: synth.cube_cloud(150, 0.3), "gauss"),
])
def test_three_body_vs_oracle(name, gen, forces, mlp2, mlp3):
    X = gen()
    N = len(X)
    F = synth.gravity_forces(N) if forces == "gravity" else synth.gaussian_forces(N)
    ctx = make_ctx(mlp2, mlp3, rcut3=4.0, ws_mb=512)
    ctx.build_tree(to_dev(X))
    ctx.build_blocks()
    U = ctx.matvec(to_dev(F), parts=8).cpu().numpy()
    Uo, nf = oracle.three_body(X, F, mlp3, 4.0, brute=(N <= 200))
    assert ctx.stats()["n_faces"] == nf                   # the fp32 cutoff decisions agree exactly (S-22)
    assert rel_l2(U, Uo) <= 1e-5
    ctx.close()


def test_full_step_c2_shape(mlp2, mlp3):
    """config-2-shaped small case: ball, gravity, two-body H-matrix + three-body + self, Euler steps with rebuild"""
    N, dt = 3000, 0.01
    X = synth.ball_cloud(N, 0.2)
    F = synth.gravity_forces(N)
    ctx = make_ctx(mlp2, mlp3, rcut3=4.0, leaf_size=32, ws_mb=1024)
    Xd = to_dev(X)
    Fd = to_dev(F)
    Xcur = X.copy()
    for step in range(3):
        Xbefore = Xd.cpu().numpy()
        assert np.array_equal(Xbefore, Xcur)
        U = ctx.step(Xd, Fd, dt=dt).cpu().numpy()
        # oracle on the positions the GPU used at this step (trajectories diverge at the 1e-6 level otherwise)
        H = oracle.HMatrix(Xbefore, mlp2, leaf=32, eta=1.0)
        replay, _ = gpu_replay(ctx, ctx.get_tree(), H)
        U2, info = H.matvec(F, f32(1e-4), replay=replay)
        U3, _ = oracle.three_body(Xbefore, F, mlp3, 4.0)
        assert rel_l2(U, U2 + U3) <= 1e-5
        # S-25: X <- X + dt U in fp32 from the GPU's own U is bit-exact
        Xcur = oracle.euler(Xbefore, U.astype(np.float64), dt)
        assert np.array_equal(Xd.cpu().numpy(), Xcur)
    ctx.close()


def test_zero_force_leaves_x_unchanged(mlp2):
    X = synth.cube_cloud(1000, 0.1)
    ctx = make_ctx(mlp2, ws_mb=512)
    Xd = to_dev(X)
    U = ctx.step(Xd, to_dev(np.zeros_like(X)), dt=0.5).cpu().numpy()
    assert np.all(U == 0) and np.array_equal(Xd.cpu().numpy(), X)
    ctx.close()


def test_step_host_matches_device_step(mlp2, mlp3):
    import torch
    N = 2500
    X = synth.cube_cloud(N, 0.1)
    F = synth.gaussian_forces(N)
    ctx = make_ctx(mlp2, mlp3, rcut3=4.0, ws_mb=1024)
    Xd = to_dev(X)
    Ud = ctx.step(Xd, to_dev(F), dt=0.01).cpu().numpy()
    Xh = torch.from_numpy(X.copy()).pin_memory()
    Fh = torch.from_numpy(F.copy()).pin_memory()
    Uh = torch.empty_like(Fh).pin_memory()
    ctx.step_host(Xh, Fh, Uh, dt=0.01)
    assert rel_l2(Uh.numpy(), Ud) <= 2e-6                 # atomics: summation order only
    assert np.max(np.abs(Xh.numpy() - Xd.cpu().numpy())) <= 1e-5
    ctx.close()


def test_self_terms_of_eq6_with_18_output_networks():
    """networks with 18 outputs [alpha^(s), alpha^(t)] (Eq. (2)).  The transverse halves feed
    the H-matrix and the three-body term as before; the self halves give the diagonal terms M^(s,2), M^(s,3) of Eq. (6)
    (L108-L113), summed over the neighbours within R_cut and applied to F_i (`parts` bit 4)."""
    n, rcut = 3000, 4.0
    X = synth.ball_cloud(n, 0.2, seed=6)
    F = synth.gaussian_forces(n, seed=7)
    m2 = synth.xavier_mlp((4, 32, 32, 18), 1, bias_scale=0.1)
    m3 = synth.xavier_mlp((7, 64, 64, 18), 3, bias_scale=0.1)
    ctx = make_ctx(m2, m3, leaf_size=32, eta=1.0, aca_tol=1e-5, rcut3=rcut, ws_mb=2048)
    ctx.build_tree(to_dev(X))
    ctx.build_blocks()
    Us = ctx.matvec(to_dev(F), parts=16).cpu().numpy()
    st = ctx.stats()
    Uo, npairs, nfaces = oracle.self_terms(X, F, m2, m3, rcut)
    assert st["n_self_pairs"] == npairs and npairs > 0 and nfaces > 0
    print("self terms: rel L2 vs oracle %.3e (%d pairs, %d faces)" % (rel_l2(Us, Uo), npairs, nfaces))
    assert rel_l2(Us, Uo) <= 1e-5
    # the transverse three-body term from the transverse half
    U3 = ctx.matvec(to_dev(F), parts=8).cpu().numpy()
    U3o, nf = oracle.three_body(X, F, m3, rcut)
    assert ctx.stats()["n_faces"] == nf == nfaces and rel_l2(U3, U3o) <= 1e-5
    # everything together against the definition, Eq. (6): alpha_1 F + M^(t,2) F (dense) + M^(s,2) F + M^(t,3) F + M^(s,3) F
    U = ctx.matvec(to_dev(F)).cpu().numpy()
    Uall = oracle.dense_matvec(X, F, m2) + U3o + Uo
    print("Eq. (6), all five terms: rel L2 vs the definition %.3e" % rel_l2(U, Uall))
    assert rel_l2(U, Uall) <= 1e-4
    ctx.close()
    # a two-body network with a self half and no three-body network at all
    ctx = make_ctx(m2, None, leaf_size=32, eta=1.0, aca_tol=1e-5, rcut3=rcut, ws_mb=1024)
    ctx.build_tree(to_dev(X))
    ctx.build_blocks()
    U2 = ctx.matvec(to_dev(F), parts=16).cpu().numpy()
    U2o, _, _ = oracle.self_terms(X, F, m2, None, rcut)
    assert rel_l2(U2, U2o) <= 1e-5
    ctx.close()
