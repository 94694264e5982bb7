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
