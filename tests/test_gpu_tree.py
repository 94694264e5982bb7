"""GPU parity: Morton order, tree, boxes, P^G, P^H are bit-exact vs the oracle."""
import numpy as np
import pytest

import oracle
import synth
from gpu_util import f32, gpu_block_table, gpu_node_table, make_ctx, to_dev

pytestmark = pytest.mark.gpu

CASES = [
    ("cube2048", lambda: synth.cube_cloud(2048, 0.1), 64, 1.0),
    ("cube5000_leaf16_eta2", lambda: synth.cube_cloud(5000, 0.1), 16, 2.0),
    ("cube3000_eta05", lambda: synth.cube_cloud(3000, 0.1), 32, 0.5),
    ("ball20000", lambda: synth.ball_cloud(20000, 0.2), 64, 1.0),
    ("chains", lambda: synth.chain_cloud(200, 50, 0.1), 64, 1.0),
    ("lattice", lambda: synth.lattice_cloud(16, 16, 8, 2.5), 8, 1.0),       # exact-equality admissibility cases
    ("line", lambda: synth.line_points(768), 3, 1.0),
    ("n1", lambda: synth.cube_cloud(1, 0.1), 64, 1.0),
    ("n3", lambda: synth.cube_cloud(3, 0.1), 1, 1.0),
    ("dups", lambda: np.repeat(synth.cube_cloud(40, 0.1), 5, axis=0), 2, 1.0),   # equal keys -> middle split
    ("ragged2049", lambda: synth.cube_cloud(2049, 0.1), 64, 1.0),
]


@pytest.mark.parametrize("name,gen,leaf,eta", CASES, ids=[c[0] for c in CASES])
def test_tree_and_blocks_bit_exact(name, gen, leaf, eta, mlp2):
    X = gen()
    H = oracle.HMatrix(X, mlp2, leaf=leaf, eta=f32(eta))
    ctx = make_ctx(mlp2, leaf_size=leaf, eta=eta, ws_mb=512)
    ctx.build_tree(to_dev(X))
    ctx.build_blocks()
    tr = ctx.get_tree()
    assert np.array_equal(tr["keys"], H.keys)
    assert np.array_equal(tr["perm"], H.perm)
    nt, bmin, bmax = gpu_node_table(tr)
    ont, obmin, obmax = H.node_table()
    assert np.array_equal(nt, ont)
    assert np.array_equal(bmin.view(np.uint32), obmin.view(np.uint32))
    assert np.array_equal(bmax.view(np.uint32), obmax.view(np.uint32))
    for which in ("G", "H"):
        t, s = ctx.get_blocks(which)
        assert np.array_equal(gpu_block_table(tr, t, s), H.block_table(which)), which
    st = ctx.stats()
    assert st["n_nodes"] == H.n_nodes and st["n_leaves"] == H.n_leaves and st["depth"] == H.depth
    assert st["n_admissible"] == H.nG and st["n_inadmissible"] == H.nH
    # tree structure the header promises: BFS numbering, children adjacent, parent/level consistent
    left, right, parent, level = tr["left"], tr["right"], tr["parent"], tr["level"]
    internal = np.nonzero(left >= 0)[0]
    assert np.array_equal(right[internal], left[internal] + 1)
    assert np.array_equal(parent[left[internal]], internal) and np.array_equal(parent[right[internal]], internal)
    assert np.array_equal(level[left[internal]], level[internal] + 1)
    assert np.all(np.diff(level) >= 0)
    ctx.close()


def test_rebuild_same_context_different_n(mlp2):
    ctx = make_ctx(mlp2, ws_mb=512)
    for n in (1000, 4000, 500):
        X = synth.cube_cloud(n, 0.1, seed=n)
        H = oracle.HMatrix(X, mlp2, leaf=64, eta=1.0)
        ctx.build_tree(to_dev(X))
        ctx.build_blocks()
        tr = ctx.get_tree()
        assert np.array_equal(tr["perm"], H.perm)
        t, s = ctx.get_blocks("G")
        assert np.array_equal(gpu_block_table(tr, t, s), H.block_table("G"))
    ctx.close()


def test_error_paths(mlp2):
    import paper_2505_08174_b200 as hh
    ctx = make_ctx(mlp2, ws_mb=512)
    with pytest.raises(hh.HHError) as e:
        ctx.build_blocks()
    assert e.value.code == -4
    with pytest.raises(hh.HHError):
        ctx.set_params(eta=-1.0)
    ctx.close()
    with pytest.raises(hh.HHError) as e:
        make_ctx(mlp2, ws_mb=1)
    assert e.value.code == -2
