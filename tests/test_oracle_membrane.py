"""Pins of the membrane oracle (oracle/membrane.py; SURVEY 8(f) NEXT-4 "with a simple membrane energy"; PAPER.md L41-43;
DESIGN.md reading A18).  -m "not gpu".  Pinned by what the formulas fix: a hand-worked spring, zero energy and gradient at
rest, central finite differences (energy -> gradient, gradient -> Hessian on stretched edges, where the clamp is inactive),
the clamp itself in closed form on one compressed edge, rigid-motion invariance, positive semi-definiteness, and the dense
matrix against the matrix-free product."""
import numpy as np


def mesh(seed=3, n=5):
    rng = np.random.default_rng(seed)
    u, v = np.meshgrid(np.linspace(0, 1, n), np.linspace(0, 1, n), indexing="ij")
    rest = np.stack([u.ravel(), v.ravel(), 0.1 * np.sin(3 * u.ravel())], axis=1)
    q = lambda i, j: i * n + j
    tr = []
    for i in range(n - 1):
        for j in range(n - 1):
            tr += [[q(i, j), q(i + 1, j), q(i + 1, j + 1)], [q(i, j), q(i + 1, j + 1), q(i, j + 1)]]
    return rest, np.array(tr, dtype=np.int32), rng


def test_hand_worked_spring_and_edge_list(oracle_mod):
    from oracle import membrane as mb
    tris = np.array([[0, 1, 2], [2, 1, 3]], dtype=np.int32)
    assert mb.edges_of(tris).tolist() == [[0, 1], [0, 2], [1, 2], [1, 3], [2, 3]]       # the shared edge once
    # one triangle, unit right-angle legs; vertex 1 pulled from (1,0,0) to (3,0,0): edge (0,1) 1 -> 3, edge (1,2) sqrt2 -> sqrt10
    rest = np.array([[0, 0, 0], [1, 0, 0], [0, 1, 0.0]])
    pos = rest.copy()
    pos[1] = [3, 0, 0]
    E, g = mb.energy_grad(pos, rest, np.array([[0, 1, 2]], dtype=np.int32), k=2.0)
    s = np.sqrt(10) - np.sqrt(2)
    assert abs(E - (0.5 * 2.0 * (2.0 ** 2 + s ** 2))) < 1e-14
    np.testing.assert_allclose(g[0], [-2.0 * 2.0, 0, 0], atol=1e-14)                   # k (|d| - L) d/|d|, d = x0 - x1 = (-3,0,0)
    np.testing.assert_allclose(g[1], [4.0 + 2.0 * s * 3 / np.sqrt(10), -2.0 * s / np.sqrt(10), 0], atol=1e-13)
    np.testing.assert_allclose(g.sum(0), 0, atol=1e-13)
    # at rest: nothing
    E0, g0 = mb.energy_grad(rest, rest, np.array([[0, 1, 2]], dtype=np.int32), 2.0)
    assert E0 == 0.0 and not g0.any()


def test_finite_differences_and_invariance(oracle_mod):
    from oracle import membrane as mb
    rest, tris, rng = mesh()
    pos = 1.6 * rest + rng.normal(scale=0.01, size=rest.shape)        # every edge stretched: the clamp is inactive
    Ed = mb.edges_of(tris)
    assert (np.linalg.norm(pos[Ed[:, 0]] - pos[Ed[:, 1]], axis=1) > np.linalg.norm(rest[Ed[:, 0]] - rest[Ed[:, 1]], axis=1)).all()
    k, h = 3.0, 1e-6
    E, g = mb.energy_grad(pos, rest, tris, k)
    gfd = np.zeros_like(pos)
    for i in range(pos.shape[0]):
        for c in range(3):
            xp, xm = pos.copy(), pos.copy()
            xp[i, c] += h
            xm[i, c] -= h
            gfd[i, c] = (mb.energy_grad(xp, rest, tris, k)[0] - mb.energy_grad(xm, rest, tris, k)[0]) / (2 * h)
    assert np.abs(g - gfd).max() <= 1e-7 * np.abs(g).max()
    p = rng.normal(size=pos.shape)
    y = mb.hess_vec(pos, rest, tris, k, p)
    yfd = (mb.energy_grad(pos + h * p, rest, tris, k)[1] - mb.energy_grad(pos - h * p, rest, tris, k)[1]) / (2 * h)
    assert np.abs(y - yfd).max() <= 1e-6 * np.abs(y).max()
    # dense matrix == matrix-free product, symmetric, PSD, translations in the null space; diagonal blocks
    H = mb.dense_hessian(pos, rest, tris, k)
    assert np.abs(H @ p.ravel() - y.ravel()).max() <= 1e-12 * np.abs(y).max()
    assert np.abs(H - H.T).max() == 0.0 and np.linalg.eigvalsh(H)[0] > -1e-10 * np.abs(H).max()
    assert np.abs(H @ np.tile([0.3, -1.0, 2.0], pos.shape[0])).max() <= 1e-12 * np.abs(H).max()
    D = mb.diag_blocks(pos, rest, tris, k)
    for v in (0, 7, 24):
        np.testing.assert_allclose(D[v], H[3 * v:3 * v + 3, 3 * v:3 * v + 3], atol=1e-13)
    # rigid motion: energy unchanged, gradient rotates
    Q, _ = np.linalg.qr(rng.normal(size=(3, 3)))
    E2, g2 = mb.energy_grad(pos @ Q.T + [1, 2, 3], rest, tris, k)
    assert abs(E2 - E) <= 1e-12 * E and np.abs(g2 - g @ Q.T).max() <= 1e-12 * np.abs(g).max()


def test_compressed_edge_clamp(oracle_mod):
    """One edge compressed to half its rest length along x: K = k n n^T exactly (the transverse part, k (1 - L/|d|) < 0, is
    clamped); stretched to twice: K = k [n n^T + (1/2)(I - n n^T)]."""
    from oracle import membrane as mb
    rest = np.array([[0, 0, 0], [1, 0, 0], [0, 5, 0.0]])
    tris = np.array([[0, 1, 2]], dtype=np.int32)
    for scale, c in ((0.5, 0.0), (2.0, 0.5)):
        pos = rest.copy()
        pos[1] = [scale, 0, 0]
        E, K = mb.edge_blocks(pos, rest, tris, 4.0)
        i = E.tolist().index([0, 1])
        np.testing.assert_allclose(K[i], 4.0 * np.diag([1.0, c, c]), atol=1e-14)
    # the clamped matrix stays PSD on a crumpled (compressed) mesh
    rest, tris, rng = mesh(seed=9)
    pos = 0.6 * rest + rng.normal(scale=0.01, size=rest.shape)
    assert np.linalg.eigvalsh(mb.dense_hessian(pos, rest, tris, 1.0))[0] > -1e-12


def test_newton_step_with_membrane(oracle_mod):
    """The combined step: direction == numpy.linalg.solve on the dense (H_T + H_m + mu I) when the inner solve converges;
    Armijo holds; with a stiff membrane the step keeps the edge lengths (relative change << without it)."""
    from oracle import membrane as mb
    from paper_2606_06511_b200 import inputs
    pb = inputs.config0_soup(n_tris=48, pool=40, seed=5)
    nV = pb.pos.shape[0]
    r = oracle_mod.assemble(pb.pos, pb.tris, pb.pairs, 1.0, 2)
    for k in (1.0, 1e3):
        s = mb.newton_step(pb.pos, pb.pos, pb.tris, pb.pairs, k, mu=1e-2, pcg_iter=600)
        H = mb._bsr_dense(r, nV) + mb.dense_hessian(pb.pos, pb.pos, pb.tris, k) + 1e-2 * np.eye(3 * nV)
        d_ref = np.linalg.solve(H, r["grad"].ravel()).reshape(nV, 3)                  # at rest g_m = 0
        assert np.linalg.norm(s["d"] - d_ref) <= 1e-8 * np.linalg.norm(d_ref)
        assert s["accepted"] and s["E1"] <= s["E0"] - 1e-4 * s["alpha"] * s["gd"] and s["E_membrane"] == 0.0
    E = mb.edges_of(pb.tris)
    def strain(x):
        return np.abs(np.linalg.norm(x[E[:, 0]] - x[E[:, 1]], axis=1) / np.linalg.norm(pb.pos[E[:, 0]] - pb.pos[E[:, 1]], axis=1) - 1).max()
    soft = mb.newton_step(pb.pos, pb.pos, pb.tris, pb.pairs, 1e-3, mu=1e-2, pcg_iter=50)
    stiff = mb.newton_step(pb.pos, pb.pos, pb.tris, pb.pairs, 1e3, mu=1e-2, pcg_iter=50)
    assert strain(stiff["x"]) < 0.05 * strain(soft["x"])


def test_no_active_pair_is_a_fixed_point_and_untangle_stops(oracle_mod):
    """Reading A16 (the loop ends when no pair is active) carried over to the membrane step: with an empty candidate list, or
    one whose pairs are all apart, x is returned unchanged and accepted -- even when the membrane itself is strained."""
    from oracle import membrane as mb
    rest, tris, rng = mesh()
    pos = 1.2 * rest
    s = mb.newton_step(pos, rest, tris, np.zeros((0, 2), dtype=np.int32), 3.0)
    assert s["accepted"] and s["n_active"] == 0 and s["alpha"] == 0.0 and (s["x"] == pos).all() and s["E_membrane"] > 0
    r = mb.untangle(pos, rest, tris, 3.0, inflate=0.0, max_steps=5)
    assert len(r["history"]) == 1 and (r["x"] == pos).all()
