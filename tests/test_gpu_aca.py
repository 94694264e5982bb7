"""GPU parity: Alg. 2 factors, far-field apply and the whole H mat-vec vs the oracle.

ACA factors are not unique (SURVEY 8(c) "several results are correct"): the oracle re-runs Alg. 2 in fp64
with the GPU's pivots and rank (replay) and checks that every GPU decision is an arg-max / a correct stop
within 1e-3 relative slack or within the running fp32 rounding bound of the residual it was taken on
(oracle replay checker); what is unique given the pivots -- each rank term C_k(i) Q_k(j), the block
product and the mat-vec -- is compared element by element."""
import numpy as np
import pytest

import oracle
import synth
from conftest import rel_l2
from gpu_util import f32, make_ctx, map_blocks_to_oracle, to_dev

pytestmark = pytest.mark.gpu


def gpu_replay(ctx, tr, H):
    """((ranks, piv_i, piv_j, flags), flags) of all GPU blocks re-ordered to the oracle's P^G order; a block on
    which Alg. 2 broke down (flag 2, S-18b) lists its attempted pivot after the accepted ones"""
    t, s = ctx.get_blocks("G")
    omap = map_blocks_to_oracle(tr, t, s, H)
    ranks, flags = ctx.get_ranks()
    pi, pj = {}, {}
    for g in range(len(t)):
        f = ctx.get_factors(g, 0, 0, want_factors=False)
        assert f["rank"] == ranks[g] and f["flag"] == flags[g] and len(f["piv_i"]) == ranks[g] + (flags[g] == 2)
        pi[omap[g]], pj[omap[g]] = f["piv_i"], f["piv_j"]
    inv = np.argsort(omap)
    r_o = ranks[inv]
    return (r_o, np.concatenate([pi[g] for g in range(len(t))]) if len(t) else np.zeros(0, np.int32),
            np.concatenate([pj[g] for g in range(len(t))]) if len(t) else np.zeros(0, np.int32), flags[inv]), flags[inv]


def setup(X, mlp, **kw):
    ctx = make_ctx(mlp, ws_mb=kw.pop("ws_mb", 1024), **kw)
    ctx.build_tree(to_dev(X))
    ctx.build_blocks()
    return ctx


@pytest.mark.parametrize("rule", [0, 1])
def test_block_factors_vs_oracle_replay(rule, mlp2):
    X = synth.cube_cloud(3000, 0.1)
    zeta = 1e-4
    H = oracle.HMatrix(X, mlp2, leaf=32, eta=2.0)
    H.set_replay_roundoff(2.0 ** -24)
    kappa = 0.0 if rule == 0 else 300.0      # Frobenius pivots (the listing's variant, S-18) reach cond 1e3..2e5: S-18b opted in
    H.set_kappa_max(kappa if kappa > 0 else float("inf"))
    ctx = setup(X, mlp2, leaf_size=32, eta=2.0, aca_tol=zeta, pivot_rule=rule, kappa_max=kappa)
    assert ctx.aca(0) == H.nG
    tr = ctx.get_tree()
    t, s = ctx.get_blocks("G")
    omap = map_blocks_to_oracle(tr, t, s, H)
    sizes = (tr["hi"][t] - tr["lo"][t]) * (tr["hi"][s] - tr["lo"][s])
    pick = list(np.argsort(-sizes)[:6]) + list(np.argsort(sizes)[:6]) + list(range(0, len(t), max(1, len(t) // 12)))
    bad_total = strict_total = n_dense = 0
    for g in pick:
        m, n = int(tr["hi"][t[g]] - tr["lo"][t[g]]), int(tr["hi"][s[g]] - tr["lo"][s[g]])
        f = ctx.get_factors(int(g), m, n)
        o = H.aca_block(int(omap[g]), zeta, rule=rule, replay=(f["piv_i"], f["piv_j"]), replay_flag=f["flag"])
        assert o["rank"] == f["rank"] and o["flag"] == f["flag"]
        bad_total += o["replay_bad"]
        strict_total += H.last_bad_strict()
        if f["flag"] == 2 or f["rank"] == 0:
            n_dense += 1                      # Alg. 2 broke down (S-18b): the block is applied densely, no factors to compare
            continue
        Cg = f["C"].reshape(-1, m, 3, 3).astype(np.float64)
        Qg = f["Q"].reshape(-1, n, 3, 3).astype(np.float64)
        Pg = np.einsum("kiab,kjbc->ijac", Cg, Qg)                  # block product sum_k C_k(i) Q_k(j)
        Po = np.einsum("kiab,kjbc->ijac", o["C"], o["Q"])
        # the fp32 bar of north_star for the primary |det| rule.  Frobenius pivots (the listing's variant, S-18)
        # sit nearer the kappa_max = 300 limit of S-18b, where fp32 entry noise is amplified most: bar 1e-4 there.
        assert rel_l2(Pg, Po) <= (1e-5 if rule == 0 else 1e-4), (g, m, n, f["rank"])
        # normalisation of the listing (L221): C_k(i_k) = I
        for k in range(f["rank"]):
            assert np.abs(Cg[k, f["piv_i"][k]] - np.eye(3)).max() <= 1e-6
        # interpolation property on the GPU's own factors: product equals G on pivot rows and columns
        G = H.dense_block(int(omap[g]))
        scale = np.abs(G).max()
        assert np.abs(Pg[f["piv_i"]] - G[f["piv_i"]]).max() <= 5e-5 * scale
        assert np.abs(Pg[:, f["piv_j"]] - G[:, f["piv_j"]]).max() <= 5e-5 * scale
    print("rule", rule, "picked blocks gone dense:", n_dense, "decisions outside the 1e-3 slack alone:", strict_total,
          "outside slack and fp32 rounding:", bad_total)
    if rule == 0:
        assert n_dense < len(pick) // 4      # Frobenius pivots (rule 1) are mostly beyond kappa_max: those blocks go dense
    assert bad_total <= 1          # see test_matvec_vs_oracle: the rounding model is first order


# Alg. 2 as printed inverts the pivot block whatever its condition: that is the default on both sides
# (kappa = 0 -> never).  Two runs of Alg. 2 with the same pivots, one on fp32 entries (relative noise ~2e-7, not
# smooth) and one on exact entries, differ by about noise x cond_F(P) on a block ("why fp32 entries
# bound the replay parity"): the plain rows report what fp32 entries achieve on the listing as printed and assert the
# north_star bar where it is met; S-18b (opt-in, kappa > 0: ill-conditioned pivots break Alg. 2 down, the block is
# applied densely) is what brings ball / chain clouds inside 1e-5.  BARS[name] = (bar on U, bar on the far-field part).
#   *_f64: aca_precision = 1 (fp64 entries and residuals in Alg. 2, factors still fp32), plain listing: the discrepancy is gone.
CASES = [
    ("c1", lambda: synth.cube_cloud(2048, 0.1), 64, 1.0, 1e-4, 0.0, 0),
    ("cube_leaf16_eta2", lambda: synth.cube_cloud(4000, 0.1), 16, 2.0, 1e-3, 0.0, 0),
    ("ball_1e-5", lambda: synth.ball_cloud(5000, 0.2), 32, 1.0, 1e-5, 0.0, 0),
    ("ball_1e-5_S18b", lambda: synth.ball_cloud(5000, 0.2), 32, 1.0, 1e-5, 300.0, 0),
    ("ball_1e-5_f64", lambda: synth.ball_cloud(5000, 0.2), 32, 1.0, 1e-5, 0.0, 1),
    ("chains", lambda: synth.chain_cloud(120, 50, 0.1), 32, 1.0, 1e-4, 0.0, 0),
    ("chains_S18b", lambda: synth.chain_cloud(120, 50, 0.1), 32, 1.0, 1e-4, 50.0, 0),
    ("chains_f64", lambda: synth.chain_cloud(120, 50, 0.1), 32, 1.0, 1e-4, 0.0, 1),
]
BARS = {"c1": (1e-5, 1e-5), "cube_leaf16_eta2": (1e-5, 1e-5), "ball_1e-5": (1e-5, 3e-5), "ball_1e-5_S18b": (1e-5, 3e-5),
        "ball_1e-5_f64": (1e-5, 1e-5), "chains": (3e-5, 1e-4), "chains_S18b": (1e-5, 1e-5), "chains_f64": (1e-5, 3e-5)}


@pytest.mark.parametrize("name,gen,leaf,eta,zeta,kappa,prec", CASES)
def test_matvec_vs_oracle(name, gen, leaf, eta, zeta, kappa, prec, mlp2):
    X = gen()
    N = len(X)
    F = synth.gaussian_forces(N)
    bar_u, bar_far = BARS[name]
    H = oracle.HMatrix(X, mlp2, leaf=leaf, eta=f32(eta))
    H.set_replay_roundoff(2.0 ** -24)
    H.set_kappa_max(kappa if kappa > 0 else float("inf"))
    ctx = setup(X, mlp2, leaf_size=leaf, eta=eta, aca_tol=zeta, kappa_max=kappa, aca_precision=prec, ws_mb=8192)
    U = ctx.matvec(to_dev(F)).cpu().numpy()
    tr = ctx.get_tree()
    st = ctx.stats()
    assert st["aca_batches"] == 1
    replay, flags = gpu_replay(ctx, tr, H)
    Uo, info = H.matvec(F, f32(zeta), replay=replay)
    # (1) the bar: GPU vs oracle with the GPU's pivots
    err = rel_l2(U, Uo)
    # far-field alone over the resident factors (row 9), against the far part of the same replay, relative to ITSELF
    Ufar = ctx.far_apply_resident(to_dev(F)).cpu().numpy()
    Uofar, _ = H.matvec(F, f32(zeta), replay=replay, include_self=False, near=False)
    err_far = rel_l2(Ufar, Uofar)
    print("%s (kappa %s): rel L2 vs replay: U %.3e, far part %.3e (|U_far| / |U| = %.2f); blocks gone dense %d of %d"
          % (name, kappa if kappa > 0 else "inf", err, err_far, np.linalg.norm(Uofar) / np.linalg.norm(Uo), st["aca_singular"], H.nG))
    assert err <= bar_u
    assert err_far <= bar_far
    if kappa == 0.0:
        # plain listing: flag 2 can only be an exactly singular pivot (|det| < 1e-30, S-18)
        diff = np.flatnonzero(info["flags"] != flags)
        for g in diff[:8]:
            print(name, "flag mismatch: oracle block", g, "shape", H.block_shape(int(g)), "GPU flag", flags[g], "replay flag", info["flags"][g],
                  "rank", replay[0][g])
        # plain listing: a flag differs only where the fp64 replay meets an exactly singular pivot block (|det| < 1e-30, S-18;
        # collinear chains produce them) that fp32 entry noise hid from the GPU; each is listed above and counted as bad
        assert np.all(info["flags"][diff] == 2) and len(diff) <= info["replay_bad"]
    else:
        # S-18b: the replay takes the GPU's breakdowns as given and judges them (plausible within a factor 2 of kappa);
        # a flag differs only where the fp64 replay meets an exactly singular pivot that fp32 noise hid from the GPU,
        # and each such block is counted as a bad decision
        assert int(np.sum(info["flags"] != flags)) <= info["replay_bad"]
    print(name, "replay decisions outside slack alone:", H.last_bad_strict(), "outside slack and fp32 rounding:", info["replay_bad"])
    # every decision is an arg-max / a correct stop / a plausible breakdown up to slack and the first-order fp32
    # rounding model (oracle/hh_oracle.cpp, K_G and K_T; K_G is pinned by test_gpu_near.py::test_entry_error_bound);
    # the model is first order, not a rigorous bound: a 2e-4 fraction of the 3 decisions per rank term may fall outside it
    assert info["replay_bad"] <= max(2, int(2e-4 * 3 * info["ranks"].sum()))
    # (2) reported: free-running oracle
    Uf, finfo = H.matvec(F, f32(zeta))
    print(name, "free-run rel L2", rel_l2(U, Uf), "rank diff blocks", int(np.sum(finfo["ranks"] != info["ranks"])))
    # (3) both within zeta of the dense product
    Ud = oracle.dense_matvec(X, F, mlp2)
    assert rel_l2(U, Ud) <= zeta and rel_l2(Uo, Ud) <= zeta
    assert st["sum_rank"] == int(replay[0].sum())
    # S-18b: blocks on which Alg. 2 broke down are counted and applied densely
    assert st["aca_singular"] == int((flags == 2).sum())
    shapes = np.array([H.block_shape(g) for g in range(H.nG)])
    assert st["fallback_entries"] == int(np.sum((flags == 2) * shapes[:, 0] * shapes[:, 1]))
    if name == "chains_S18b":
        print(name, "dense fraction of blocks: %.3f" % (st["aca_singular"] / H.nG))
    ctx.close()


def test_far_apply_kernel_vs_its_own_factors(mlp2):
    """row 9 in isolation: k_far over the resident factors against sum_k C_k (Q_k F^sigma) evaluated in fp64 from the SAME
    factors (fetched through hh_get_factors), relative to the far-field part itself: the apply kernel's own fp32 error"""
    X = synth.cube_cloud(3000, 0.1, seed=5)
    N = len(X)
    F = synth.gaussian_forces(N)
    ctx = setup(X, mlp2, leaf_size=32, eta=2.0, aca_tol=1e-4)
    nG = ctx.stats()["n_admissible"]
    assert ctx.aca(0) == nG
    tr = ctx.get_tree()
    t, s = ctx.get_blocks("G")
    Fs = F[tr["perm"]].astype(np.float64)
    Us = np.zeros((N, 3))
    for g in range(nG):
        lo_t, hi_t, lo_s, hi_s = int(tr["lo"][t[g]]), int(tr["hi"][t[g]]), int(tr["lo"][s[g]]), int(tr["hi"][s[g]])
        f = ctx.get_factors(g, hi_t - lo_t, hi_s - lo_s)
        if f["flag"] == 2 or f["rank"] == 0:
            continue
        Cg = f["C"].reshape(-1, hi_t - lo_t, 3, 3).astype(np.float64)
        Qg = f["Q"].reshape(-1, hi_s - lo_s, 3, 3).astype(np.float64)
        tk = np.einsum("kjab,jb->ka", Qg, Fs[lo_s:hi_s])
        Us[lo_t:hi_t] += np.einsum("kiab,kb->ia", Cg, tk)
    Uref = np.zeros((N, 3))
    Uref[tr["perm"]] = Us
    Ufar = ctx.far_apply_resident(to_dev(F)).cpu().numpy()
    err = rel_l2(Ufar, Uref)
    print("k_far vs fp64 evaluation of its own factors: rel L2 %.3e over %d blocks" % (err, nG))
    assert err <= 2e-6
    ctx.close()


@pytest.mark.parametrize("leaf,n,eta,tol", [(200, 12000, 1.0, 1e-4), (100, 9000, 1.0, 1e-5), (40, 6000, 2.0, 1e-4), (3, 700, 1.0, 1e-6),
                                             (64, 40000, 0.6, 1e-5), (250, 30000, 1.0, 1e-4)])
def test_far_ring_kernel_equals_one_cta_per_block(mlp2, leaf, n, eta, tol):
    """row 9, both forms on the SAME resident factors: the ring kernel (persistent CTAs, TMA bulk copies into a shared-memory
    byte ring; blocks with max(m,n) <= 256) against round 1's one-CTA-per-block kernel, in every ring size class (leaf 200:
    129..256, leaf 100: 65..128, leaf 40: <= 64, leaf 3: rows and columns below the pad width, ranks up to min(m,n)) and the
    whole-block ring kernel k_far_mid for 256 < max(m,n) <= 1024 (40,000 and 30,000 particles: blocks of
    300..1,000 rows, several chunks per block)"""
    X = synth.ball_cloud(n, 0.2, seed=11) if leaf != 40 else synth.chain_cloud(n // 50, 50, 0.1)
    F = synth.gaussian_forces(len(X), seed=3)
    ctx = setup(X, mlp2, leaf_size=leaf, eta=eta, aca_tol=tol)
    nG = ctx.stats()["n_admissible"]
    assert nG > 0
    first, worst = 0, 0.0
    while first < nG:                                               # every arena batch (the rank prediction may cut the first one short)
        nxt = ctx.aca(first)
        assert nxt > first
        ctx.set_far_impl(1)
        U1 = ctx.far_apply_resident(to_dev(F)).cpu().numpy()
        ctx.set_far_impl(0)
        U0 = ctx.far_apply_resident(to_dev(F)).cpu().numpy()
        U0b = ctx.far_apply_resident(to_dev(F)).cpu().numpy()      # the item list is reused while the factors stay resident
        ctx.set_far_impl(2)                                         # without k_far_mid (256 < max(m,n) <= 1024 by one CTA per block)
        U2 = ctx.far_apply_resident(to_dev(F)).cpu().numpy()
        assert np.linalg.norm(U1) > 0
        worst = max(worst, rel_l2(U0, U1), rel_l2(U0b, U1), rel_l2(U2, U1))
        first = nxt
    print("leaf %d: ring vs one-CTA-per-block far-field apply: rel L2 %.3e over %d blocks" % (leaf, worst, nG))
    assert worst <= 1e-6
    ctx.close()


def test_arena_batches_give_same_result(mlp2):
    X = synth.cube_cloud(6000, 0.1)
    F = synth.gaussian_forces(6000)
    big = setup(X, mlp2, leaf_size=16, eta=2.0, aca_tol=1e-4, ws_mb=8192)
    U1 = big.matvec(to_dev(F)).cpu().numpy()
    st1 = big.stats()
    assert st1["aca_batches"] == 1
    need = st1["workspace_required"]
    small = setup(X, mlp2, leaf_size=16, eta=2.0, aca_tol=1e-4, ws_mb=(need >> 20) + 8)   # ~72 MB of arena
    U2 = small.matvec(to_dev(F)).cpu().numpy()
    st2 = small.stats()
    assert st2["aca_batches"] > 2, st2
    assert abs(st2["sum_rank"] - st1["sum_rank"]) <= 0.002 * st1["sum_rank"]     # Gram sums are float atomics: a near-tie stop may move by one
    assert rel_l2(U2, U1) <= 2e-6
    big.close(); small.close()


def test_rank_cap_is_flagged_not_an_error(mlp2):
    X = synth.cube_cloud(3000, 0.1)
    F = synth.gaussian_forces(3000)
    H = oracle.HMatrix(X, mlp2, leaf=32, eta=1.0)
    ctx = setup(X, mlp2, leaf_size=32, eta=1.0, aca_tol=1e-6, aca_max_rank=3)
    U = ctx.matvec(to_dev(F)).cpu().numpy()
    ranks, flags = ctx.get_ranks()
    assert ranks.max() <= 3 and (flags == 1).sum() > 0
    assert ctx.stats()["aca_not_converged"] == int((flags == 1).sum())
    replay, fl = gpu_replay(ctx, ctx.get_tree(), H)
    Uo, info = H.matvec(F, f32(1e-6), max_rank=3, replay=replay)
    assert rel_l2(U, Uo) <= 1e-5
    assert np.array_equal(info["flags"], fl)
    ctx.close()


def test_degenerate_blocks(mlp2):
    """1 x q, c x 1 and 1 x 1 admissible blocks (S-15, S-21): leaf 1 on a tiny cloud"""
    X = synth.cube_cloud(40, 0.01)
    F = synth.gaussian_forces(40)
    H = oracle.HMatrix(X, mlp2, leaf=1, eta=1.0)
    ctx = setup(X, mlp2, leaf_size=1, eta=1.0, aca_tol=1e-4)
    U = ctx.matvec(to_dev(F)).cpu().numpy()
    Ud = oracle.dense_matvec(X, F, mlp2)
    assert rel_l2(U, Ud) <= 1e-4
    ranks, _ = ctx.get_ranks()
    tr = ctx.get_tree()
    t, s = ctx.get_blocks("G")
    one = np.minimum(tr["hi"][t] - tr["lo"][t], tr["hi"][s] - tr["lo"][s]) == 1
    _, flags = ctx.get_ranks()
    # one step reproduces a 1 x q / c x 1 block exactly, unless its only pivot is ill-conditioned (S-18b: dense)
    assert one.any() and np.all((ranks[one] == 1) | (flags[one] == 2)) and np.any(ranks[one] == 1)
    ctx.close()


def test_both_aca_forms_agree(mlp2):
    """hh_set_aca_impl: the lock-step forms (0, the default: entries and vectorised update in separate launches; 2: stored terms
    staged by TMA bulk copies; 3: entries and update fused; 4: form 0 on two half-batches one listing line apart, the update of one
    beside the entry evaluation of the other) and the one-CTA-per-block form (1) run the same Alg. 2; pivots, ranks
    and flags agree on all but near-tie blocks and the mat-vecs agree to fp32 summation order.  The lock-step forms do the same
    arithmetic in the same order on each entry (only the Gram sums are float atomics), so they differ by even less."""
    X = synth.cube_cloud(5000, 0.1, seed=9)
    F = synth.gaussian_forces(5000)
    res = []
    for impl in (0, 1, 2, 3, 4):
        ctx = setup(X, mlp2, leaf_size=32, eta=1.0, aca_tol=1e-4, ws_mb=8192)
        ctx.set_aca_impl(impl)
        U = ctx.matvec(to_dev(F)).cpu().numpy()
        ranks, flags = ctx.get_ranks()
        res.append((U, ranks, flags, ctx.stats()))
        ctx.close()
    U0, r0, f0, s0 = res[0]
    for impl in (1, 2, 3, 4):
        U1, r1, f1, s1 = res[impl]
        assert s0["aca_batches"] == s1["aca_batches"] == 1
        print("aca_impl %d vs 0: rel L2 %.3e, ranks differ on %.4f of the blocks" % (impl, rel_l2(U0, U1), np.mean(r0 != r1)))
        lim = 0.02 if impl == 1 else 0.005
        assert np.mean(r0 != r1) < lim and np.mean(f0 != f1) < lim
        assert rel_l2(U0, U1) <= 1e-5


IMPLS = (0, 2, 3, 4)


@pytest.mark.parametrize("name,gen,leaf,eta,zeta", [
    ("ball_tol1e-6_ranks_beyond_staging", lambda: synth.ball_cloud(6000, 0.2, seed=4), 48, 1.0, 1e-6),
    ("big_blocks_slices", lambda: synth.cube_cloud(20000, 0.1, seed=6), 64, 0.7, 1e-4),
    ("tiny_leaves", lambda: synth.cube_cloud(1500, 0.1, seed=8), 5, 1.0, 1e-5),
])
def test_lockstep_forms_agree(mlp2, name, gen, leaf, eta, zeta):
    """the three lock-step forms against each other -- k2_eval + k2_upd (default: 4 rows resp. 2 columns per thread, vector loads),
    k2_step_t (tiles of 256 rows, the first 10 stored terms staged by TMA), k2_step (fused, one entry per thread) -- on clouds that
    exercise: ranks beyond the staged 10, slices of blocks larger than a tile and blocks that straddle a tile boundary, leaves
    smaller than a granule (pad rows and columns inside a thread's vector)"""
    X = gen()
    F = synth.gaussian_forces(len(X), seed=5)
    out = []
    for impl in IMPLS:
        ctx = setup(X, mlp2, leaf_size=leaf, eta=eta, aca_tol=zeta, ws_mb=8192)
        ctx.set_aca_impl(impl)
        U = ctx.matvec(to_dev(F)).cpu().numpy()
        ranks, flags = ctx.get_ranks()
        out.append((U, ranks, flags))
        ctx.close()
    U0, r0, f0 = out[0]
    for impl, (U2, r2, f2) in zip(IMPLS[1:], out[1:]):
        print(name, "aca_impl %d vs 0: rel L2 %.3e, max rank %d, ranks differ on %.4f of %d blocks" % (impl, rel_l2(U0, U2), r0.max(), np.mean(r0 != r2), len(r0)))
        assert np.mean(r0 != r2) < 0.005 and np.mean(f0 != f2) < 0.005
        assert rel_l2(U0, U2) <= 10 * zeta * 0.01 + 2e-6


def test_arena_overflow_is_retried_with_a_smaller_batch(mlp2):
    """ranks far above the first batch's prediction (32) overflow the arena in the middle of the lock-step loop; the batch
    is then shrunk and run again (hh_aca2.cu), and the mat-vec equals the one computed with plenty of space"""
    X = synth.cube_cloud(4000, 0.1, seed=21)
    F = synth.gaussian_forces(4000)
    big = setup(X, mlp2, leaf_size=32, eta=2.0, aca_tol=1e-7, ws_mb=16384)
    U1 = big.matvec(to_dev(F)).cpu().numpy()
    st1 = big.stats()
    ranks1, _ = big.get_ranks()
    assert st1["aca_batches"] == 1 and ranks1.max() > 40
    need = st1["workspace_required"]
    small = setup(X, mlp2, leaf_size=32, eta=2.0, aca_tol=1e-7, ws_mb=(need >> 20) + 40 + (st1["factor_bytes"] >> 20) // 3)
    U2 = small.matvec(to_dev(F)).cpu().numpy()
    st2 = small.stats()
    assert st2["aca_batches"] >= 3, st2
    assert st2["n_admissible"] == st1["n_admissible"]
    assert abs(st2["sum_rank"] - st1["sum_rank"]) <= 0.002 * st1["sum_rank"]       # Gram sums are atomics: near-tie stops may differ
    assert rel_l2(U2, U1) <= 5e-6
    big.close(); small.close()
