"""Pins of the oracle's EXACT Hessian (second-order forward duals through App. A; SURVEY 8(f) NEXT-3,
second half -- the terms PAPER.md L26 "ignores").  -m "not gpu".  Pinned by calculus and algebra, not by itself:
central finite differences of the FIRST-order gradient (which has its own pins), the chain-rule identity
H_exact = H_EQ4 + 2 tc0 tc1^2 d2tc0 + 2 tc1 tc0^2 d2tc1, Euler's identity for a degree-4 homogeneous function
(H_exact x = 3 grad), symmetry, translation / rotation invariance, and the worked example's first-order values."""
import numpy as np
import pytest


def random_active_pairs(oracle, n, seed):
    rng = np.random.default_rng(seed)
    out = []
    while len(out) < n:
        x = rng.random(18)
        r = oracle.pair(x, 1.0, 0)
        if r["active"] and np.abs(r["tc"]).min() > 1e-2:
            out.append(x)
    return out


def test_first_order_part_equals_the_first_order_oracle(oracle_mod):
    """value, tc and gradient of the second-order evaluation == the (separately pinned) first-order oracle; worked example A."""
    xa = np.array([-1, -1, 0, 3, -1, 0, 1, 1, 0, 0, 0, -1, 4, 0, -1, 2, 0, 1], dtype=float)
    e = oracle_mod.pair_exact(xa)
    assert e["active"] and np.allclose(e["tc"], [-3, 1], atol=1e-14) and abs(e["energy"] - 9) < 1e-13
    np.testing.assert_allclose(e["grad"], [-3, 3, -3, 9, 9, -9, 6, 12, -12, -9, -9, 9, 3, -3, 3, -6, -12, 12], atol=1e-12)
    for x in random_active_pairs(oracle_mod, 20, 1):
        e, r = oracle_mod.pair_exact(x), oracle_mod.pair(x, 1.0, 0)
        np.testing.assert_allclose(e["tc"], r["tc"], rtol=1e-13)
        np.testing.assert_allclose(e["grad"], r["grad"], rtol=1e-11, atol=1e-13 * np.abs(r["grad"]).max())
    # separated pair: inactive, all zero
    far = xa.copy()
    far[9:] += 10.0
    e = oracle_mod.pair_exact(far)
    assert not e["active"] and not e["H"].any() and not e["grad"].any()


def test_chain_rule_identity_and_symmetry(oracle_mod):
    """H_exact - H_EQ4 = 2 tc0 tc1^2 H0 + 2 tc1 tc0^2 H1 (the dropped terms), all matrices symmetric."""
    for x in random_active_pairs(oracle_mod, 20, 2):
        e, r = oracle_mod.pair_exact(x), oracle_mod.pair(x, 1.0, 0)
        tc0, tc1 = e["tc"]
        drop = 2 * tc0 * tc1 ** 2 * e["H0"] + 2 * tc1 * tc0 ** 2 * e["H1"]
        scale = np.abs(e["H"]).max()
        assert np.abs(e["H"] - r["H"] - drop).max() <= 1e-11 * scale
        for M in (e["H"], e["H0"], e["H1"]):
            assert np.abs(M - M.T).max() <= 1e-11 * max(np.abs(M).max(), 1e-300)
        assert np.abs(drop).max() > 1e-3 * scale          # the dropped part is not negligible


def test_finite_differences_of_the_gradient(oracle_mod):
    """Column j of H_exact (H0, H1) == central difference of grad (g0, g1) along x_j."""
    h = 1e-6
    for x in random_active_pairs(oracle_mod, 6, 3):
        e = oracle_mod.pair_exact(x)
        Hfd, H0fd, H1fd = np.zeros((18, 18)), np.zeros((18, 18)), np.zeros((18, 18))
        for j in range(18):
            xp, xm = x.copy(), x.copy()
            xp[j] += h
            xm[j] -= h
            rp, rm = oracle_mod.pair(xp, 1.0, 0), oracle_mod.pair(xm, 1.0, 0)
            assert rp["active"] and rm["active"]
            Hfd[:, j] = (rp["grad"] - rm["grad"]) / (2 * h)
            H0fd[:, j] = (rp["g0"] - rm["g0"]) / (2 * h)
            H1fd[:, j] = (rp["g1"] - rm["g1"]) / (2 * h)
        for M, F in ((e["H"], Hfd), (e["H0"], H0fd), (e["H1"], H1fd)):
            assert np.abs(M - F).max() <= 2e-6 * np.abs(M).max(), np.abs(M - F).max() / np.abs(M).max()


def test_homogeneity_and_invariance(oracle_mod):
    """T is homogeneous of degree 4 and invariant under rigid motion: H x = 3 grad; H (1 (x) c) = 0;
    d2tc_r x = 0 (tc is homogeneous of degree 1); rotating the pair rotates the blocks."""
    rng = np.random.default_rng(4)
    for x in random_active_pairs(oracle_mod, 10, 4):
        e = oracle_mod.pair_exact(x)
        s = np.abs(e["H"]).max() * np.abs(x).max()
        assert np.abs(e["H"] @ x - 3 * e["grad"]).max() <= 1e-10 * s
        assert np.abs(e["H0"] @ x).max() <= 1e-10 * np.abs(e["H0"]).max() and np.abs(e["H1"] @ x).max() <= 1e-10 * np.abs(e["H1"]).max()
        c = np.tile(rng.normal(size=3), 6)
        assert np.abs(e["H"] @ c).max() <= 1e-10 * np.abs(e["H"]).max()
        Q, _ = np.linalg.qr(rng.normal(size=(3, 3)))
        R = np.kron(np.eye(6), Q)
        e2 = oracle_mod.pair_exact(R @ x + np.tile(rng.normal(size=3), 6))
        assert np.abs(e2["H"] - R @ e["H"] @ R.T).max() <= 1e-9 * np.abs(e["H"]).max()


def test_exact_hess_vec_sums_the_pairs(oracle_mod):
    from paper_2606_06511_b200 import inputs
    pb = inputs.config0_soup()
    p = np.random.default_rng(5).normal(size=pb.pos.shape)
    y = oracle_mod.exact_hess_vec(pb.pos, pb.tris, pb.pairs, p)
    ref = np.zeros_like(pb.pos)
    for pr in pb.pairs:
        vid = np.concatenate([pb.tris[pr[0]], pb.tris[pr[1]]])
        e = oracle_mod.pair_exact(pb.pos[vid].ravel())
        if e["active"]:
            np.add.at(ref, vid, (e["H"] @ p[vid].ravel()).reshape(6, 3))
    assert np.linalg.norm(y - ref) <= 1e-12 * np.linalg.norm(ref)
    # y(x) = 3 grad (Euler), summed over pairs
    g = oracle_mod.assemble(pb.pos, pb.tris, pb.pairs, 1.0, 0, want_hess=False)["grad"]
    yx = oracle_mod.exact_hess_vec(pb.pos, pb.tris, pb.pairs, pb.pos)
    assert np.linalg.norm(yx - 3 * g) <= 1e-9 * np.linalg.norm(3 * g)


def test_exact_assembly_against_dense(oracle_mod):
    """assemble(hess_mode=HESS_EXACT): the BSR equals a dense 576 x 576 accumulation of pair_exact's matrices written in
    the test (shared-vertex variant included), the pattern is the Eq. 4 pattern, BSR.p == exact_hess_vec(p), and Euler's
    identity H x = 3 grad holds for the assembled matrix."""
    from paper_2606_06511_b200 import inputs
    for pb in (inputs.config0_soup(), inputs.config0_soup(n_tris=48, pool=40, seed=5)):
        nV = pb.pos.shape[0]
        r = oracle_mod.assemble(pb.pos, pb.tris, pb.pairs, 1.0, oracle_mod.HESS_EXACT)
        r0 = oracle_mod.assemble(pb.pos, pb.tris, pb.pairs, 1.0, oracle_mod.HESS_EQ4)
        assert (r["rowptr"] == r0["rowptr"]).all() and (r["colind"] == r0["colind"]).all()
        np.testing.assert_array_equal(r["grad"], r0["grad"])
        D = np.zeros((3 * nV, 3 * nV))
        for pr in pb.pairs:
            vid = np.concatenate([pb.tris[pr[0]], pb.tris[pr[1]]])
            if len(set(vid.tolist())) < 6:
                continue
            e = oracle_mod.pair_exact(pb.pos[vid].ravel())
            if e["active"]:
                idx = (3 * vid[:, None] + np.arange(3)[None, :]).ravel()
                D[np.ix_(idx, idx)] += e["H"]
        B = np.zeros_like(D)
        for v in range(nV):
            for k in range(r["rowptr"][v], r["rowptr"][v + 1]):
                c = r["colind"][k]
                B[3 * v:3 * v + 3, 3 * c:3 * c + 3] = r["vals"][k]
        assert np.abs(B - D).max() <= 1e-12 * np.abs(D).max()
        assert np.abs(B - B.T).max() <= 1e-11 * np.abs(B).max()
        p = np.random.default_rng(6).normal(size=pb.pos.shape)
        y = oracle_mod.bsr_matvec(r["rowptr"], r["colind"], r["vals"], p)
        ye = oracle_mod.exact_hess_vec(pb.pos, pb.tris, pb.pairs, p)
        assert np.linalg.norm(y - ye) <= 1e-12 * np.linalg.norm(ye)
        yx = oracle_mod.bsr_matvec(r["rowptr"], r["colind"], r["vals"], pb.pos)
        assert np.linalg.norm(yx - 3 * r["grad"]) <= 1e-9 * np.linalg.norm(3 * r["grad"])
        # the exact matrix really differs from Eq. 4 (the dropped terms are not small)
        assert np.linalg.norm(r["vals"] - r0["vals"]) > 1e-2 * np.linalg.norm(r0["vals"])
