"""Pins of the oracle's consumer loop (oracle/newton.py; SURVEY 8(f) NEXT-2 "line search on tt_energy" and NEXT-4;
PAPER.md L5, L41-43; reading A16).  -m "not gpu".  The step is pinned by what the textbook fixes, not by
itself: the Newton direction against LAPACK's solve of the dense shifted system built from the (separately pinned)
per-pair Hessian, the gradient-descent limit mu -> infinity in closed form, the Armijo rule re-evaluated by brute force
over the whole step-length sequence, monotone descent, and the end state of an untangling run classified by the
edge-pierces-triangle test of test_oracle_pins.py (not Moeller's)."""
import numpy as np

from test_oracle_pins import _brute_force_intersects

XA = np.array([-1, -1, 0, 3, -1, 0, 1, 1, 0, 0, 0, -1, 4, 0, -1, 2, 0, 1], dtype=float)   # worked example A: tc = (-3, 1), T = 9


def one_pair():
    pos = XA.reshape(6, 3).copy()
    tris = np.array([[0, 1, 2], [3, 4, 5]], dtype=np.int32)
    pairs = np.array([[0, 1]], dtype=np.int32)
    return pos, tris, pairs


def test_direction_is_the_shifted_newton_direction(oracle_mod):
    """d = (H + mu I)^-1 g: PCG run to convergence == numpy.linalg.solve on the dense 18 x 18 system."""
    from oracle import newton
    pos, tris, pairs = one_pair()
    for mode in (2, 3):
        pr = oracle_mod.pair(XA, 1.0, mode)
        for mu in (1.0, 1e-2):
            s = newton.newton_step(pos, tris, pairs, hess_mode=mode, mu=mu, pcg_iter=200, pcg_rtol=1e-15)
            d_ref = np.linalg.solve(pr["H"] + mu * np.eye(18), pr["grad"])
            assert np.linalg.norm(s["d"].ravel() - d_ref) <= 1e-10 * np.linalg.norm(d_ref)
            assert abs(s["gd"] - pr["grad"] @ d_ref) <= 1e-10 * abs(pr["grad"] @ d_ref)
            assert s["E0"] == 9.0 and s["gd"] > 0          # a descent direction: x moves along -d


def test_gradient_descent_limit(oracle_mod):
    """mu -> infinity: d = g / mu + O(|H| |g| / mu^2), and a full step x - d is accepted (tiny, so Armijo holds)."""
    from oracle import newton
    pos, tris, pairs = one_pair()
    pr = oracle_mod.pair(XA, 1.0, 2)
    mu = 1e6
    s = newton.newton_step(pos, tris, pairs, hess_mode=2, mu=mu, pcg_iter=50, pcg_rtol=1e-15)
    g = pr["grad"]
    assert np.linalg.norm(s["d"].ravel() - g / mu) <= 2 * np.linalg.norm(pr["H"], 2) * np.linalg.norm(g) / mu ** 2
    assert s["accepted"] and s["alpha"] == 1.0 and s["backtracks"] == 0
    np.testing.assert_allclose(s["x"], pos - s["d"], rtol=0, atol=0)
    # first-order decrease: E1 = E0 - g.d + O(|d|^2)
    assert abs((s["E0"] - s["E1"]) - s["gd"]) <= 1e-3 * s["gd"]


def test_armijo_rule_by_brute_force(oracle_mod):
    """The accepted alpha is the FIRST of 1, 1/2, 1/4, ... that satisfies Armijo; energies recomputed pair by pair."""
    from oracle import newton
    from paper_2606_06511_b200 import inputs
    pb = inputs.config0_soup()
    c1 = 1e-4
    for mu in (1e-3, 1e-1):
        s = newton.newton_step(pb.pos, pb.tris, pb.pairs, hess_mode=2, mu=mu, pcg_iter=20, c1=c1)
        assert s["accepted"] and s["gd"] > 0
        def E(x):
            tot = 0.0
            for pr in pb.pairs:
                tot += oracle_mod.pair(x[np.concatenate([pb.tris[pr[0]], pb.tris[pr[1]]])].ravel(), 1.0, 0)["energy"]
            return tot
        E0 = E(pb.pos)
        assert abs(E0 - s["E0"]) <= 1e-12 * E0
        alpha, j = 1.0, 0
        while True:
            ok = E(pb.pos - alpha * s["d"]) <= E0 - c1 * alpha * s["gd"]
            if ok:
                break
            alpha *= 0.5
            j += 1
        assert alpha == s["alpha"] and j == s["backtracks"]
        assert s["E1"] < s["E0"]


def test_untangling_two_crossing_sheets(oracle_mod):
    """Two small triangulated sheets pushed through each other: the energy falls monotonically and the loop ends with NO
    intersecting pair according to the brute-force classifier (6 edge-pierces-triangle tests per pair, not Moeller)."""
    from oracle import newton
    rng = np.random.default_rng(5)
    n = 4
    u, v = np.meshgrid(np.linspace(0, 1, n), np.linspace(0, 1, n), indexing="ij")
    quad = lambda i, j: i * n + j
    tr = []
    for i in range(n - 1):
        for j in range(n - 1):
            tr += [[quad(i, j), quad(i + 1, j), quad(i + 1, j + 1)], [quad(i, j), quad(i + 1, j + 1), quad(i, j + 1)]]
    tr = np.array(tr, dtype=np.int32)
    a = np.stack([u.ravel(), v.ravel(), 0.06 * np.sin(3 * u.ravel())], axis=1)
    b = np.stack([u.ravel() + 0.013, v.ravel() + 0.021, 0.02 - 0.05 * np.sin(3 * u.ravel() + 0.4)], axis=1)
    pos = np.concatenate([a, b]) + rng.normal(scale=1e-3, size=(2 * n * n, 3))
    tris = np.concatenate([tr, tr + n * n]).astype(np.int32)
    cand0 = oracle_mod.broad_phase(pos, tris, 0.05)
    assert oracle_mod.pairs(pos, tris, cand0, 1.0, want_J=False)["active"].sum() >= 4
    r = newton.untangle(pos, tris, inflate=0.05, max_steps=60, hess_mode=2, mu=1e-2, pcg_iter=30)
    h = r["history"]
    assert all(s["accepted"] for s in h)
    assert all(h[i]["E1"] <= h[i]["E0"] for i in range(len(h)))
    assert h[-1]["n_active"] == 0, [s["n_active"] for s in h]
    x = r["x"]
    nT = tris.shape[0]
    for i in range(nT):
        for j in range(i + 1, nT):
            if set(tris[i]) & set(tris[j]):
                continue
            assert not _brute_force_intersects(x[tris[i]], x[tris[j]]), (i, j)
