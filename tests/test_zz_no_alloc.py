"""hh_dense_matvec_static: the ONE entry point that allocates nothing (include/hh.h, csrc/hh_static.cu) -- scratch in a
file-scope static __device__ array, no context, no workspace, N <= HH_STATIC_MAX_N.

Checked against the EXISTING path: hh_matvec with nothing admissible (eta -> 0+: every block near-field),
self + near-field parts, at the tolerance the near-field tests use (relative L2 <= 1e-5), on two calls in a row with
different clouds and sizes (the static array keeps the first call's contents: nothing stale may leak into the second).

This file is collected last (pytest -x: a failure here must not hide other tests) and passes alone in a
fresh process as well as after the other tests."""
import numpy as np
import pytest

import synth
from conftest import rel_l2
from gpu_util import make_ctx, to_dev

pytestmark = pytest.mark.gpu


def existing_path(X, F, mlp):
    ctx = make_ctx(mlp, leaf_size=64, eta=1e-30, ws_mb=512)
    ctx.build_tree(to_dev(X))
    ctx.build_blocks()
    assert ctx.stats()["n_admissible"] == 0
    U = ctx.matvec(to_dev(F), parts=3).cpu().numpy()          # self term + near-field = the dense product
    ctx.close()
    return U


def test_static_entry_point_matches_existing_path_twice_in_a_row(mlp2_bias):
    import torch
    import paper_2505_08174_b200 as hh
    cases = [(synth.cube_cloud(3000, 0.1, seed=31), synth.gaussian_forces(3000, seed=32)),
             (synth.ball_cloud(1777, 0.2, seed=33), synth.gaussian_forces(1777, seed=34))]
    refs = [existing_path(X, F, mlp2_bias) for X, F in cases]
    dm = hh.DeviceMlp(mlp2_bias)
    dev = [(to_dev(X), to_dev(F), torch.empty(len(X), 3, dtype=torch.float32, device="cuda")) for X, F in cases]
    hh.dense_matvec_static(dm, dev[0][0], dev[0][1], out=dev[0][2])      # first call on this device: looks up the array's address
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    hh.dense_matvec_static(dm, dev[1][0], dev[1][1], out=dev[1][2])      # second call, smaller cloud, straight after
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 == free0, "the call changed the device's free memory: something allocated"
    U = [d[2].cpu().numpy() for d in dev]
    for k in range(2):
        err = rel_l2(U[k], refs[k])
        print("call %d (N = %d): static entry point vs hh_matvec (nothing admissible): rel L2 %.3e" % (k + 1, len(refs[k]), err))
        assert np.isfinite(U[k]).all()
        assert err <= 1e-5
    # the first cloud again, after the smaller one: same bits as the first time (fixed summation order, nothing stale)
    again = hh.dense_matvec_static(dm, dev[0][0], dev[0][1]).cpu().numpy()
    assert np.array_equal(again, U[0])


def test_static_entry_point_rejects_sizes_beyond_its_scratch(mlp2_bias, mlp3):
    import torch
    import paper_2505_08174_b200 as hh
    dm = hh.DeviceMlp(mlp2_bias)
    n = hh.STATIC_MAX_N + 1
    X = torch.zeros(n, 3, dtype=torch.float32, device="cuda")
    with pytest.raises(hh.HHError) as e:
        hh.dense_matvec_static(dm, X, X)
    assert e.value.code == -2 and "HH_STATIC_MAX_N" in str(e.value)
    with pytest.raises(hh.HHError) as e:                                 # only the 4-32-32-9 two-body network
        hh.dense_matvec_static(hh.DeviceMlp(mlp3), X[:10], X[:10])
    assert e.value.code == -5
    # the largest size is accepted
    Xm = to_dev(synth.cube_cloud(hh.STATIC_MAX_N, 0.1, seed=35))
    U = hh.dense_matvec_static(dm, Xm, to_dev(synth.gaussian_forces(hh.STATIC_MAX_N, seed=36)))
    assert bool(torch.isfinite(U).all())
