"""Pins of the oracle's block-Jacobi preconditioner and conjugate gradients (
PAPER.md L5 names an "inexact Newton optimization route" and nothing else, so the operations are their
textbook definitions).  -m "not gpu".  Each pin is something other than the oracle itself: hand
arithmetic (tests/golden/pcg_example.txt), LAPACK (numpy.linalg.inv / solve / eigvalsh), and the theorems
of CG (finite termination, monotone energy-norm error, residual recurrence)."""
import os

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def golden():
    out = {}
    for line in open(os.path.join(ROOT, "tests", "golden", "pcg_example.txt")):
        if line.startswith("#") or not line.strip():
            continue
        f = line.split()
        out[f[0]] = np.array([float(v) for v in f[1:]])
    return out


def lifted_2x2():
    rp = np.array([0, 2, 4], dtype=np.int32)
    ci = np.array([0, 1, 0, 1], dtype=np.int32)
    I = np.eye(3)
    vals = np.stack([4 * I, 1 * I, 1 * I, 3 * I])
    b = np.array([[1.0, 1, 1], [2, 2, 2]])
    return rp, ci, vals, b


def dense_of(rp, ci, vals, nV):
    H = np.zeros((3 * nV, 3 * nV))
    for r in range(nV):
        for e in range(rp[r], rp[r + 1]):
            H[3 * r:3 * r + 3, 3 * ci[e]:3 * ci[e] + 3] += vals[e]
    return H


@pytest.fixture(scope="module")
def soup_system(oracle_mod):
    """Config 0's assembled PSD2 Hessian (always PSD; singular: translations, untouched vertices) and its gradient."""
    from paper_2606_06511_b200 import inputs
    pb = inputs.config0_soup()
    ref = oracle_mod.assemble(pb.pos, pb.tris, pb.pairs, 1.0, oracle_mod.HESS_PSD2)
    return pb, ref


def test_hand_example(oracle_mod):
    g = golden()
    rp, ci, vals, b = lifted_2x2()
    r = oracle_mod.pcg(rp, ci, vals, b, 0.0, 5, 1e-14, precond=False, history=True)
    assert r["iters"] == 2                                            # two distinct eigenvalues: exact in two steps
    for c in range(3):
        np.testing.assert_allclose(r["x_hist"][1][:, c], g["x1_plain"], rtol=0, atol=1e-15)
        np.testing.assert_allclose(r["x"][:, c], g["x_exact"], rtol=0, atol=1e-15)
    r = oracle_mod.pcg(rp, ci, vals, b, 0.0, 5, 1e-14, precond=True, history=True)
    assert r["iters"] == 2
    for c in range(3):
        np.testing.assert_allclose(r["x_hist"][1][:, c], g["x1_jacobi"], rtol=0, atol=1e-15)
        np.testing.assert_allclose(r["x"][:, c], g["x_exact"], rtol=0, atol=1e-15)
    np.testing.assert_allclose(r["minv"][0], np.eye(3) / 4, atol=1e-16)
    np.testing.assert_allclose(r["minv"][1], np.eye(3) / 3, atol=1e-16)
    # shift: (A + 2 I) x = b -> [[6,1],[1,5]]^-1 [1,2] = [3/29, 11/29]
    r = oracle_mod.pcg(rp, ci, vals, b, 2.0, 5, 1e-14)
    np.testing.assert_allclose(r["x"][:, 0], [3 / 29, 11 / 29], atol=1e-15)


def test_block_jacobi_against_lapack(oracle_mod, soup_system):
    pb, ref = soup_system
    nV = pb.n_verts
    for shift in (1e-3, 0.5):
        minv = oracle_mod.block_jacobi(ref["rowptr"], ref["colind"], ref["vals"], shift)
        H = dense_of(ref["rowptr"], ref["colind"], ref["vals"], nV)
        for v in range(nV):
            blk = H[3 * v:3 * v + 3, 3 * v:3 * v + 3] + shift * np.eye(3)
            np.testing.assert_allclose(minv[v], np.linalg.inv(blk), rtol=1e-9, atol=1e-12 * np.abs(np.linalg.inv(blk)).max())
    # a vertex no active pair touches has the block shift * I
    untouched = np.nonzero(np.diff(ref["rowptr"]) == 0)[0]
    if untouched.size:
        np.testing.assert_allclose(minv[untouched[0]], np.eye(3) / 0.5, atol=1e-15)
    # a general (non-symmetric, needs pivoting) block: [[0,2,0],[1,0,0],[0,0,4]]^-1 = [[0,1,0],[.5,0,0],[0,0,.25]]
    rp = np.array([0, 1], dtype=np.int32)
    ci = np.array([0], dtype=np.int32)
    m = oracle_mod.block_jacobi(rp, ci, np.array([[[0, 2, 0], [1, 0, 0], [0, 0, 4.0]]]), 0.0)
    np.testing.assert_allclose(m[0], [[0, 1, 0], [0.5, 0, 0], [0, 0, 0.25]], atol=1e-16)


@pytest.mark.parametrize("precond", [False, True])
def test_converges_to_dense_solve(oracle_mod, soup_system, precond):
    """(H + mu I) x = -grad on config 0 (576 unknowns) against numpy.linalg.solve; the energy-norm error
    decreases monotonically (the defining optimality property of CG) and the recurred residual equals b - A x_k."""
    pb, ref = soup_system
    nV = pb.n_verts
    H = dense_of(ref["rowptr"], ref["colind"], ref["vals"], nV)
    assert np.linalg.eigvalsh(0.5 * (H + H.T))[0] > -1e-9 * np.abs(H).max()          # PSD2 is PSD
    mu = 1e-2 * np.trace(H) / (3 * nV)
    A = H + mu * np.eye(3 * nV)
    b = -ref["grad"]
    x_star = np.linalg.solve(A, b.ravel())
    r = oracle_mod.pcg(ref["rowptr"], ref["colind"], ref["vals"], b, mu, 1000, 1e-13, precond=precond, history=True)
    assert r["iters"] < 1000
    assert np.linalg.norm(r["x"].ravel() - x_star) <= 1e-9 * np.linalg.norm(x_star)
    err = [float((xk.ravel() - x_star) @ A @ (xk.ravel() - x_star)) for xk in r["x_hist"]]
    assert all(e1 <= e0 * (1 + 1e-9) for e0, e1 in zip(err[:-1], err[1:]))
    assert err[-1] <= 1e-18 * err[0]
    for k in (1, 5, r["iters"] // 2):
        rk = b.ravel() - A @ r["x_hist"][k].ravel()
        assert abs(np.linalg.norm(rk) - r["res"][k]) <= 1e-8 * r["res"][0]
    assert r["res"][-1] <= 1e-13 * np.linalg.norm(b)


def test_finite_termination_three_eigenvalues(oracle_mod):
    """CG reaches the exact solution in as many steps as A has distinct eigenvalues (here 3: 1, 2, 5)."""
    rng = np.random.default_rng(5)
    nV = 4
    Q, _ = np.linalg.qr(rng.normal(size=(12, 12)))
    A = Q @ np.diag([1.0] * 5 + [2.0] * 4 + [5.0] * 3) @ Q.T
    rp = np.arange(0, 4 * nV + 1, 4, dtype=np.int32)[:nV + 1]
    ci = np.tile(np.arange(nV, dtype=np.int32), nV)
    vals = np.stack([A[3 * r:3 * r + 3, 3 * c:3 * c + 3] for r in range(nV) for c in range(nV)])
    b = rng.normal(size=(nV, 3))
    r = oracle_mod.pcg(rp, ci, vals, b, 0.0, 10, 1e-12, precond=False)
    assert r["iters"] == 3
    np.testing.assert_allclose(r["x"].ravel(), np.linalg.solve(A, b.ravel()), rtol=1e-10, atol=1e-12)


def test_stopping_rule(oracle_mod, soup_system):
    pb, ref = soup_system
    b = -ref["grad"]
    r = oracle_mod.pcg(ref["rowptr"], ref["colind"], ref["vals"], b, 0.1, 500, 1e-4)
    assert r["iters"] < 500 and r["res"][-1] <= 1e-4 * np.linalg.norm(b) < r["res"][-2]
    r5 = oracle_mod.pcg(ref["rowptr"], ref["colind"], ref["vals"], b, 0.1, 5, 0.0)
    assert r5["iters"] == 5 and r5["res"].shape[0] == 6            # rtol 0: exactly max_iter steps
