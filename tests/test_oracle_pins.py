"""Pins for the CPU oracle (-m "not gpu").  Each test checks oracle/ against something that is
NOT the oracle: a hand-worked fixture (tests/golden/), a closed form, an invariant, central
finite differences, a textbook brute-force routine, or a Monte-Carlo constant.  Citations are
PAPER.md lines; P*/I*/A* labels are DESIGN.md's."""
import os

import numpy as np
import pytest

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def load_fixture(name):
    out = {}
    with open(os.path.join(GOLD, name)) as f:
        for line in f:
            line = line.split("#")[0].strip()
            if not line:
                continue
            k, v = line.split(":")
            out[k.strip()] = np.array([float(t) for t in v.split()])
    return out


def x_of(fx):
    return np.concatenate([fx["a"], fx["b"]])


def rand_active_pairs(oracle, n, seed, margin=1e-3):
    """Random uniform-[0,1]^3 pairs that the oracle calls active and that sit >= margin away
    from every discrete boundary we can see from outside (|tc|, FD-stable)."""
    rng = np.random.default_rng(seed)
    out = []
    while len(out) < n:
        x = rng.random(18)
        r = oracle.pair(x, 1.0, oracle.HESS_EQ4)
        if not r["active"] or min(abs(r["tc"])) < margin:
            continue
        # stay clear of kinks: the same pair perturbed a little must keep a smooth tc
        ok = True
        for _ in range(4):
            xp = x + 2e-5 * rng.normal(size=18)
            rp = oracle.pair(xp, 1.0, oracle.HESS_EQ4)
            if not rp["active"] or np.abs(rp["tc"] - r["tc"]).max() > 1e-2 * np.abs(r["tc"]).min() + 1e-3:
                ok = False
        if ok:
            out.append(x)
    return out


# ---------------------------------------------------------------- P1 / P2: hand-worked examples
@pytest.mark.parametrize("name", ["example_A.txt", "example_B.txt"])
def test_worked_examples(oracle_mod, name):
    fx = load_fixture(name)
    r = oracle_mod.pair(x_of(fx), 1.0, oracle_mod.HESS_EQ4)
    assert r["active"] == bool(fx["active"][0])
    np.testing.assert_allclose(r["tc"], fx["tc"], rtol=0, atol=1e-14)        # Eq. 1
    np.testing.assert_allclose(r["energy"], fx["energy"][0], rtol=1e-14)     # Eq. 2
    np.testing.assert_allclose(r["g0"], fx["g0"], rtol=0, atol=1e-13)
    np.testing.assert_allclose(r["g1"], fx["g1"], rtol=0, atol=1e-13)
    np.testing.assert_allclose(r["lam"], fx["lam"], rtol=1e-13)              # L47
    if "grad" in fx:
        np.testing.assert_allclose(r["grad"], fx["grad"], rtol=0, atol=1e-12)   # Eq. 3
    if "H_a0a0" in fx:
        np.testing.assert_allclose(r["H"][0:3, 0:3].ravel(), fx["H_a0a0"], atol=1e-12)   # Eq. 4
        np.testing.assert_allclose(r["H"][0:3, 9:12].ravel(), fx["H_a0b0"], atol=1e-12)
        w = np.linalg.eigvalsh(r["H"])
        np.testing.assert_allclose([w[0], w[-1]], fx["eig_EQ4"], rtol=1e-9)
        assert np.abs(w[1:-1]).max() < 1e-12                                   # rank 2
        np.testing.assert_allclose(np.linalg.norm(r["H"]), fx["frob_EQ4"][0], rtol=1e-7)
        h2 = oracle_mod.pair(x_of(fx), 1.0, oracle_mod.HESS_PSD2)["H"]
        np.testing.assert_allclose(np.linalg.norm(h2), fx["frob_PSD2"][0], rtol=1e-7)
        p3 = r["H"] - h2                                                       # third part alone
        w3 = np.linalg.eigvalsh(p3)
        np.testing.assert_allclose([w3[0], w3[-1]], fx["eig_part3"], rtol=1e-6)
        np.testing.assert_allclose(np.trace(p3), fx["lam"][2], rtol=1e-12)     # A7: L47 prints the trace


def test_filter_mode_keeps_or_drops_third_part(oracle_mod):
    """A7: FILTER keeps part 3 iff L47's third quantity >= 0 (example A keeps, B drops)."""
    for name, keep in (("example_A.txt", True), ("example_B.txt", False)):
        x = x_of(load_fixture(name))
        e = oracle_mod.pair(x, 1.0, oracle_mod.HESS_EQ4)["H"]
        f = oracle_mod.pair(x, 1.0, oracle_mod.HESS_FILTER)["H"]
        p = oracle_mod.pair(x, 1.0, oracle_mod.HESS_PSD2)["H"]
        np.testing.assert_allclose(f, e if keep else p, atol=1e-13)
        assert np.linalg.eigvalsh(p)[0] > -1e-12                               # parts 1+2 are PSD (L47)


def test_sigma_half_reproduces_listing_scale(oracle_mod):
    """A6: App. A L154-155 multiplies tc by 0.5: tc halves, T, grad, H scale by exactly 1/16."""
    x = x_of(load_fixture("example_A.txt"))
    r1 = oracle_mod.pair(x, 1.0, oracle_mod.HESS_EQ4)
    rh = oracle_mod.pair(x, 0.5, oracle_mod.HESS_EQ4)
    np.testing.assert_allclose(rh["tc"], [-1.5, 0.5], atol=1e-15)
    np.testing.assert_allclose(rh["energy"], 9.0 / 16.0, rtol=1e-15)
    np.testing.assert_allclose(rh["grad"], r1["grad"] / 16.0, atol=1e-14)
    np.testing.assert_allclose(rh["H"], r1["H"] / 16.0, atol=1e-14)
    assert rh["active"] == r1["active"]


# ---------------------------------------------------------------- P3: shift family
@pytest.mark.parametrize("s", [-3.0, -2.5, -2.0, -1.0, 0.0, 0.5, 1.0, 1.5, -3.5])
def test_shift_family(oracle_mod, s):
    """Example A with T_b translated by (s,0,0): I_b = [1+s, 3+s] so tc = (-3-s, 1-s);
    T(s) = ((3+s)(1-s))^2 inside (-3,1), exactly 0 outside and on the boundary (L13-17)."""
    fx = load_fixture("example_A.txt")
    b = fx["b"].reshape(3, 3) + np.array([s, 0, 0])
    r = oracle_mod.pair(np.concatenate([fx["a"], b.ravel()]), 1.0, oracle_mod.HESS_EQ4)
    if -3.0 < s < 1.0:
        assert r["active"]
        np.testing.assert_allclose(r["tc"], [-3 - s, 1 - s], atol=1e-14)
        np.testing.assert_allclose(r["energy"], ((3 + s) * (1 - s)) ** 2, rtol=1e-13)
    else:
        assert not r["active"]
        assert r["energy"] == 0.0 and not r["grad"].any() and not r["H"].any()


# ---------------------------------------------------------------- P4: separated / excluded pairs
def test_separated_and_excluded_pairs(oracle_mod):
    fx = load_fixture("example_A.txt")
    a = fx["a"]
    far = fx["b"].reshape(3, 3) + np.array([0, 0, 10.0])          # all of b on one side of plane(a)
    coplanar = fx["a"].reshape(3, 3) + np.array([0.5, 0.25, 0.0])  # same plane z=0 (L11 excludes)
    degenerate = np.array([[0, 0, -1], [0, 0, -1], [2, 0, 1.0]])   # zero-area triangle
    for b in (far, coplanar, degenerate):
        r = oracle_mod.pair(np.concatenate([a, b.ravel()]), 1.0, oracle_mod.HESS_EQ4)
        assert not r["active"] and r["energy"] == 0.0
        assert not r["grad"].any() and not r["H"].any()
    # assembly level: no active pair -> zero energy, zero gradient, empty BSR; adjacent pair dropped
    pos = np.concatenate([a.reshape(3, 3), far, [[5.0, 5.0, 5.0]]])
    tris = np.array([[0, 1, 2], [3, 4, 5], [2, 6, 4]], dtype=np.int32)
    out = oracle_mod.assemble(pos, tris, np.array([[0, 1], [0, 2]], dtype=np.int32))
    assert out["energy"] == 0.0 and not out["grad"].any() and out["nnzb"] == 0


def test_topologically_adjacent_pair_is_inactive(oracle_mod):
    """L11 / A9: triangles sharing a vertex INDEX are skipped even if they cross geometrically."""
    fx = load_fixture("example_A.txt")
    pos = np.concatenate([fx["a"].reshape(3, 3), fx["b"].reshape(3, 3)])
    crossing = oracle_mod.assemble(pos, np.array([[0, 1, 2], [3, 4, 5]], dtype=np.int32),
                                   np.array([[0, 1]], dtype=np.int32))
    assert crossing["active"][0] == 1
    pos2 = pos.copy()
    pos2[3] = pos2[0]                                              # same position, distinct index: not adjacent
    r2 = oracle_mod.pairs(pos2, np.array([[0, 1, 2], [3, 4, 5]], dtype=np.int32), np.array([[0, 1]], dtype=np.int32))
    shared = oracle_mod.pairs(pos, np.array([[0, 1, 2], [0, 4, 5]], dtype=np.int32), np.array([[0, 1]], dtype=np.int32))
    assert shared["active"][0] == 0 and shared["energy"] == 0.0
    assert r2["active"][0] in (0, 1)                               # legal input either way


# ---------------------------------------------------------------- A4: vertex exactly on the plane
def test_vertex_on_plane_branch(oracle_mod):
    """App. A: (+,-,0) -> segment0 is the on-plane vertex itself.  b2=(1,0,0) lies on
    plane(a) (z=0); b0b1 crosses it at (3,0,0): I_b=[1,3], I_a=[0,2] -> tc=(-3,1), T=9."""
    a = np.array([-1, -1, 0, 3, -1, 0, 1, 1, 0.0])
    b = np.array([0, 0, -1, 6, 0, 1, 1, 0, 0.0])
    x = np.concatenate([a, b])
    r = oracle_mod.pair(x, 1.0, oracle_mod.HESS_EQ4)
    assert r["active"]
    np.testing.assert_allclose(r["tc"], [-3, 1], atol=1e-14)
    # derivatives along directions that keep b2 exactly on plane(a): a's and b2's x,y; all of b0,b1
    free = [0, 1, 3, 4, 6, 7] + list(range(9, 15)) + [15, 16]
    h = 1e-6
    for i in free:
        xp, xm = x.copy(), x.copy()
        xp[i] += h
        xm[i] -= h
        tp = oracle_mod.pair(xp, 1.0, 0)["tc"]
        tm = oracle_mod.pair(xm, 1.0, 0)["tc"]
        fd = (tp - tm) / (2 * h)
        np.testing.assert_allclose([r["g0"][i], r["g1"][i]], fd, atol=2e-8)


# ---------------------------------------------------------------- P6: finite differences
def test_finite_differences(oracle_mod):
    """g0, g1 (the Gauss-Newton terms of Eq. 4) and Eq. 3's gradient vs central differences."""
    for x in rand_active_pairs(oracle_mod, 25, seed=7):
        r = oracle_mod.pair(x, 1.0, oracle_mod.HESS_EQ4)
        h = 1e-6
        fd_tc = np.zeros((18, 2))
        fd_T = np.zeros(18)
        for i in range(18):
            xp, xm = x.copy(), x.copy()
            xp[i] += h
            xm[i] -= h
            rp = oracle_mod.pair(xp, 1.0, 0)
            rm = oracle_mod.pair(xm, 1.0, 0)
            fd_tc[i] = (rp["tc"] - rm["tc"]) / (2 * h)
            fd_T[i] = (rp["energy"] - rm["energy"]) / (2 * h)
        scale = max(np.abs(r["g0"]).max(), np.abs(r["g1"]).max())
        np.testing.assert_allclose(r["g0"], fd_tc[:, 0], atol=2e-7 * scale)
        np.testing.assert_allclose(r["g1"], fd_tc[:, 1], atol=2e-7 * scale)
        np.testing.assert_allclose(r["grad"], fd_T, atol=2e-6 * np.abs(r["grad"]).max())


# ---------------------------------------------------------------- P5: invariants I1-I7
def _rot(rng):
    q, _ = np.linalg.qr(rng.normal(size=(3, 3)))
    if np.linalg.det(q) < 0:
        q[:, 0] = -q[:, 0]
    return q


def test_invariants(oracle_mod):
    rng = np.random.default_rng(11)
    for x in rand_active_pairs(oracle_mod, 20, seed=3):
        r = oracle_mod.pair(x, 1.0, oracle_mod.HESS_EQ4)
        X = x.reshape(6, 3)
        g0, g1 = r["g0"].reshape(6, 3), r["g1"].reshape(6, 3)
        tol = 1e-10
        # I1 rigid motion
        R, c = _rot(rng), rng.normal(size=3)
        rr = oracle_mod.pair((X @ R.T + c).ravel(), 1.0, 0)
        np.testing.assert_allclose(rr["tc"], r["tc"], rtol=tol, atol=1e-13)
        np.testing.assert_allclose(rr["energy"], r["energy"], rtol=1e-9)
        np.testing.assert_allclose(rr["grad"].reshape(6, 3), r["grad"].reshape(6, 3) @ R.T, atol=tol * np.abs(r["grad"]).max())
        Rb = np.kron(np.eye(6), R)
        np.testing.assert_allclose(rr["H"], Rb @ r["H"] @ Rb.T, atol=1e-9 * np.abs(r["H"]).max())
        # I2 swap T_a <-> T_b: tc individually unchanged
        rs = oracle_mod.pair(np.concatenate([x[9:], x[:9]]), 1.0, 0)
        np.testing.assert_allclose(rs["tc"], r["tc"], rtol=tol, atol=1e-13)
        np.testing.assert_allclose(rs["grad"], np.concatenate([r["grad"][9:], r["grad"][:9]]), atol=tol * np.abs(r["grad"]).max())
        # I3 odd relabelling of one triangle: (tc0,tc1) -> (-tc1,-tc0); T, grad unchanged
        xo = np.concatenate([X[[1, 0, 2]].ravel(), x[9:]])
        ro = oracle_mod.pair(xo, 1.0, 0)
        np.testing.assert_allclose(ro["tc"], [-r["tc"][1], -r["tc"][0]], rtol=tol, atol=1e-13)
        np.testing.assert_allclose(ro["grad"].reshape(6, 3)[[1, 0, 2, 3, 4, 5]], r["grad"].reshape(6, 3), atol=tol * np.abs(r["grad"]).max())
        # I4 uniform scale
        s = 3.7
        rk = oracle_mod.pair(s * x, 1.0, 0)
        np.testing.assert_allclose(rk["tc"], s * r["tc"], rtol=tol)
        np.testing.assert_allclose(rk["g0"], r["g0"], atol=tol * np.abs(r["g0"]).max())
        np.testing.assert_allclose(rk["energy"], s ** 4 * r["energy"], rtol=1e-9)
        np.testing.assert_allclose(rk["grad"], s ** 3 * r["grad"], rtol=1e-7, atol=tol * s ** 3 * np.abs(r["grad"]).max())
        np.testing.assert_allclose(rk["H"], s ** 2 * r["H"], atol=1e-9 * s ** 2 * np.abs(r["H"]).max())
        # I5 translation / rotation / Euler (tc is homogeneous of degree 1)
        for g, t in ((g0, r["tc"][0]), (g1, r["tc"][1])):
            gs = np.abs(g).max()
            assert np.abs(g.sum(0)).max() < tol * gs
            assert np.abs(np.cross(X, g).sum(0)).max() < tol * gs * 10
            np.testing.assert_allclose((g * X).sum(), t, rtol=1e-9, atol=1e-12)
        # I6 grad.x = 4T ; H_EQ4 x = 3 grad ; H (1 (x) c) = 0 ; symmetric ; rank <= 2
        np.testing.assert_allclose(r["grad"] @ x, 4 * r["energy"], rtol=1e-9)
        np.testing.assert_allclose(r["H"] @ x, 3 * r["grad"], atol=1e-9 * np.abs(r["grad"]).max())
        assert np.abs(r["H"] @ np.tile(c, 6)).max() < 1e-9 * np.abs(r["H"]).max()
        assert np.abs(r["H"] - r["H"].T).max() <= 4e-16 * np.abs(r["H"]).max()
        sv = np.linalg.svd(r["H"], compute_uv=False)
        assert sv[2] < 1e-12 * sv[0]
        # I7 L47's first two quantities are the non-zero eigenvalues of parts one and two
        c00, c11 = 2 * r["tc"][1] ** 2, 2 * r["tc"][0] ** 2
        np.testing.assert_allclose(np.linalg.eigvalsh(c00 * np.outer(r["g0"], r["g0"]))[-1], r["lam"][0], rtol=1e-10)
        np.testing.assert_allclose(np.linalg.eigvalsh(c11 * np.outer(r["g1"], r["g1"]))[-1], r["lam"][1], rtol=1e-10)
        # Eq. 4 is exactly J^T M J with M = [[2tc1^2, 4tc0tc1],[4tc0tc1, 2tc0^2]] (L26-33)
        J = np.stack([r["g0"], r["g1"]])
        M = np.array([[c00, 4 * r["tc"][0] * r["tc"][1]], [4 * r["tc"][0] * r["tc"][1], c11]])
        np.testing.assert_allclose(r["H"], J.T @ M @ J, atol=1e-12 * np.abs(r["H"]).max())
        # Eq. 3
        np.testing.assert_allclose(r["grad"], 2 * r["tc"][0] * r["tc"][1] ** 2 * r["g0"] + 2 * r["tc"][1] * r["tc"][0] ** 2 * r["g1"],
                                   atol=1e-13 * np.abs(r["grad"]).max())


# ---------------------------------------------------------------- P11: printed forms agree
def test_printed_forms_agree(oracle_mod):
    rng = np.random.default_rng(5)
    pos = rng.random((600, 3))
    tris = np.arange(600, dtype=np.int32).reshape(-1, 3)
    i, j = np.triu_indices(200, 1)
    prs = np.stack([i, j], 1).astype(np.int32)[:5000]
    r = oracle_mod.pairs(pos, tris, prs)
    act = r["active"].astype(bool)
    tc0, tc1 = r["tc"][act, 0], r["tc"][act, 1]
    assert ((tc0 < 0) & (tc1 > 0)).all()                                   # L15 <=> L153 on active pairs
    first_form = ((0 - (tc0 + tc1) / 2) ** 2 - ((tc1 - tc0) / 2) ** 2) ** 2   # Eq. 2, left form (L17)
    np.testing.assert_allclose(r["T"][act], first_form, rtol=1e-9)
    np.testing.assert_allclose(r["T"][act], (tc0 * tc1) ** 2, rtol=1e-14)
    assert (r["T"][~act] == 0).all() and (r["tc"][~act] == 0).all()        # A11
    # L15's own inequality (0 - mid)^2 < half^2 holds exactly for the active pairs
    assert (((tc0 + tc1) / 2) ** 2 < ((tc1 - tc0) / 2) ** 2).all()
    np.testing.assert_allclose(r["energy"], r["T"].sum(), rtol=1e-12)


# ---------------------------------------------------------------- P7: brute-force classification
def _brute_force_intersects(A, B):
    """Textbook test, independent of Moeller: two non-coplanar triangles intersect iff an edge of
    one pierces the other.  Piercing solved as a 3x3 linear system p + s(q-p) = t0 + u e1 + v e2."""
    def pierces(p, q, T):
        Mx = np.stack([q - p, -(T[1] - T[0]), -(T[2] - T[0])], axis=1)
        if abs(np.linalg.det(Mx)) < 1e-300:
            return False
        s, u, v = np.linalg.solve(Mx, T[0] - p)
        return (0 < s < 1) and (u > 0) and (v > 0) and (u + v < 1)
    for k in range(3):
        if pierces(A[k], A[(k + 1) % 3], B) or pierces(B[k], B[(k + 1) % 3], A):
            return True
    return False


def test_brute_force_classification_config0(oracle_mod):
    """Moeller's "if and only if" (L11): oracle active set == brute force on all pairs of config 0."""
    from paper_2606_06511_b200 import inputs
    pb = inputs.config0_soup()
    r = oracle_mod.pairs(pb.pos, pb.tris, pb.pairs, want_J=False)
    ref = np.array([_brute_force_intersects(pb.pos[pb.tris[i]], pb.pos[pb.tris[j]]) for i, j in pb.pairs])
    assert (ref == r["active"].astype(bool)).all()
    assert 0.2 < ref.mean() < 0.4                                           # "~30 % intersecting"
    # shared-vertex variant: adjacency rule drops pairs before geometry
    pb2 = inputs.config0_soup(n_tris=40, pool=30, seed=99)
    i, j = np.triu_indices(40, 1)
    allp = np.stack([i, j], 1).astype(np.int32)
    r2 = oracle_mod.pairs(pb2.pos, pb2.tris, allp, want_J=False)
    for (ti, tj), a in zip(allp, r2["active"]):
        if set(pb2.tris[ti]) & set(pb2.tris[tj]):
            assert a == 0


# ---------------------------------------------------------------- P8: Monte-Carlo constant
def test_monte_carlo_intersection_probability(oracle_mod):
    """Two triangles with i.i.d. uniform [0,1]^3 vertices intersect with p = 0.276 +- 0.003."""
    rng = np.random.default_rng(2024)
    n = 200_000
    pos = rng.random((6 * n, 3))
    tris = np.arange(6 * n, dtype=np.int32).reshape(-1, 3)
    prs = np.stack([np.arange(0, 2 * n, 2), np.arange(1, 2 * n, 2)], 1).astype(np.int32)
    p = oracle_mod.pairs(pos, tris, prs, want_J=False)["active"].mean()
    assert abs(p - 0.276) < 0.005


# ---------------------------------------------------------------- P9 / P10: assembly
@pytest.mark.parametrize("mode", [0, 1, 2, 3])
def test_assembly_against_dense(oracle_mod, mode):
    """BSR of config 0 (192 block rows) == dense 576x576 accumulation of the per-pair 18x18;
    H.p three ways; with p = x and EQ4, H x = 3 grad (I6)."""
    from paper_2606_06511_b200 import inputs
    for pb in (inputs.config0_soup(), inputs.config0_soup(n_tris=48, pool=40, seed=5)):
        out = oracle_mod.assemble(pb.pos, pb.tris, pb.pairs, 1.0, mode)
        nV = pb.n_verts
        Hd = np.zeros((3 * nV, 3 * nV))
        gd = np.zeros(3 * nV)
        E = 0.0
        pattern = set()
        for k, (ti, tj) in enumerate(pb.pairs):
            vid = np.concatenate([pb.tris[ti], pb.tris[tj]])
            r = oracle_mod.pair(pb.pos[vid].ravel(), 1.0, mode)
            if not r["active"]:
                continue
            E += r["energy"]
            dof = (3 * vid[:, None] + np.arange(3)).ravel()
            Hd[np.ix_(dof, dof)] += r["H"]
            gd[dof] += r["grad"]
            pattern |= {(int(p), int(q)) for p in vid for q in vid}
        np.testing.assert_allclose(out["energy"], E, rtol=1e-12)
        np.testing.assert_allclose(out["grad"].ravel(), gd, atol=1e-11 * np.abs(gd).max())
        # pattern: sorted unique, full
        got = set()
        for rrow in range(nV):
            cols = out["colind"][out["rowptr"][rrow]:out["rowptr"][rrow + 1]]
            assert (np.diff(cols) > 0).all()
            got |= {(rrow, int(c)) for c in cols}
        assert got == pattern and out["nnzb"] == len(pattern)
        Hb = np.zeros_like(Hd)
        for rrow in range(nV):
            for e in range(out["rowptr"][rrow], out["rowptr"][rrow + 1]):
                c = out["colind"][e]
                Hb[3 * rrow:3 * rrow + 3, 3 * c:3 * c + 3] = out["vals"][e]
        np.testing.assert_allclose(Hb, Hd, atol=1e-11 * np.abs(Hd).max())
        rng = np.random.default_rng(1)
        p = rng.normal(size=(nV, 3))
        y1 = oracle_mod.hess_vec_pairs(nV, pb.tris, pb.pairs, out["active"], out["tc"], out["J"], p, mode)
        y2 = oracle_mod.bsr_matvec(out["rowptr"], out["colind"], out["vals"], p)
        y3 = (Hd @ p.ravel()).reshape(nV, 3)
        np.testing.assert_allclose(y1, y3, atol=1e-11 * np.abs(y3).max())
        np.testing.assert_allclose(y2, y3, atol=1e-11 * np.abs(y3).max())
        if mode == 0:
            yx = oracle_mod.hess_vec_pairs(nV, pb.tris, pb.pairs, out["active"], out["tc"], out["J"], pb.pos, mode)
            np.testing.assert_allclose(yx, 3 * out["grad"], atol=1e-10 * np.abs(out["grad"]).max())


def test_psd_projection_mode(oracle_mod):
    """hess_mode 3: the per-pair Hessian is the PSD projection of Eq. 4's matrix.
    Pins: (a) worked example A by hand -- the non-zero eigenvalues of J^T M J are those of M G with
    G = J J^T = [[15/4, -3/4], [-3/4, 11/4]], M = [[2, -12], [-12, 18]]: trace 75, determinant
    det M det G = (-108)(39/4) = -1053, so lambda = (75 +- sqrt(9837)) / 2 and H+ is rank one with
    Frobenius norm = trace = lambda_+; (b) LAPACK's eigh (numpy) of the oracle's own Eq. 4 matrix on
    random active pairs (the oracle uses its own Jacobi sweeps); (c) H+ is symmetric, PSD, keeps the
    translation null space, H+ - H_EQ4 is PSD, and H+ = H for a matrix that is PSD already (PSD2)."""
    x = x_of(load_fixture("example_A.txt"))
    lam_p = (75.0 + np.sqrt(9837.0)) / 2.0
    lam_m = (75.0 - np.sqrt(9837.0)) / 2.0
    H3 = oracle_mod.pair(x, 1.0, 3)["H"]
    H0 = oracle_mod.pair(x, 1.0, 0)["H"]
    np.testing.assert_allclose(np.linalg.norm(H3), lam_p, rtol=1e-12)
    np.testing.assert_allclose(np.trace(H3), lam_p, rtol=1e-12)
    np.testing.assert_allclose(np.trace(H3 - H0), -lam_m, rtol=1e-11)
    w = np.linalg.eigvalsh(H3)
    assert w[0] > -1e-12 * lam_p and abs(w[-2]) < 1e-12 * lam_p                 # PSD, rank one
    rng = np.random.default_rng(33)
    seen = 0
    while seen < 40:
        xr = rng.uniform(0, 1, 18)
        r0 = oracle_mod.pair(xr, 1.0, 0)
        if not r0["active"]:
            continue
        seen += 1
        H3 = oracle_mod.pair(xr, 1.0, 3)["H"]
        lam, U = np.linalg.eigh(r0["H"])
        ref = (U * np.maximum(lam, 0.0)) @ U.T
        sc = np.abs(r0["H"]).max()
        np.testing.assert_allclose(H3, ref, atol=1e-11 * sc)
        np.testing.assert_allclose(H3, H3.T, atol=1e-13 * sc)
        assert np.linalg.eigvalsh(H3)[0] > -1e-11 * sc
        assert np.linalg.eigvalsh(H3 - r0["H"])[0] > -1e-11 * sc
        shift = np.tile(rng.normal(size=3), 6)
        assert np.abs(H3 @ shift).max() < 1e-10 * sc * np.abs(shift).max()
    # a matrix that is PSD already is its own projection: parts one and two only
    xa = x_of(load_fixture("example_A.txt"))
    r2 = oracle_mod.pair(xa, 1.0, 2)
    lam, U = np.linalg.eigh(r2["H"])
    assert lam[0] > -1e-12 * lam[-1]


def test_broad_phase_oracle(oracle_mod):
    """NEXT-1: candidate pairs = non-adjacent triangle pairs whose inflated AABBs overlap.
    Pins: hand cases (overlap, touching boxes are closed intervals, a gap closes exactly when
    2 * inflate reaches it, shared-vertex pairs dropped), lexicographic uniqueness, and agreement
    with the generators' uniform-grid routine (a different algorithm) on a mesh and a soup."""
    from paper_2606_06511_b200 import inputs
    tri = np.array([[0, 0, 0], [1, 0, 0], [0, 1, 0]], dtype=np.float64)
    def two(shift, inflate, share=False):
        pos = np.concatenate([tri, tri + np.asarray(shift, dtype=np.float64)])
        tris = np.array([[0, 1, 2], [3, 4, 5]], dtype=np.int32)
        if share:
            tris[1, 0] = 0
        return oracle_mod.broad_phase(pos, tris, inflate)
    assert two((0.5, 0.5, 0.0), 0.0).tolist() == [[0, 1]]
    assert two((1.0, 0.0, 0.0), 0.0).tolist() == [[0, 1]]            # boxes touch: closed intervals
    assert two((1.5, 0.0, 0.0), 0.0).shape[0] == 0                   # gap 0.5
    assert two((1.5, 0.0, 0.0), 0.2).shape[0] == 0                   # 2 * 0.2 < 0.5
    assert two((1.5, 0.0, 0.0), 0.25).tolist() == [[0, 1]]           # 2 * 0.25 = 0.5 (exact in binary)
    assert two((0.0, 0.0, 3.0), 0.0).shape[0] == 0                   # separated along z only
    assert two((0.5, 0.5, 0.0), 0.0, share=True).shape[0] == 0       # shares vertex 0: adjacent
    rng = np.random.default_rng(8)
    soup_pos = rng.uniform(0, 1, (1500, 3)) * np.array([1.0, 1.0, 0.2])
    soup_pos[1::3] = soup_pos[0::3] + rng.normal(0, 0.03, (500, 3))
    soup_pos[2::3] = soup_pos[0::3] + rng.normal(0, 0.03, (500, 3))
    soup_tris = np.arange(1500, dtype=np.int32).reshape(500, 3)
    ico = inputs.config1_icospheres(subdiv=3)
    for pos, tris, inflate in ((soup_pos, soup_tris, 0.0), (soup_pos, soup_tris, 0.01), (ico.pos, ico.tris, 0.02)):
        pr = oracle_mod.broad_phase(pos, tris, inflate)
        key = pr[:, 0].astype(np.int64) * tris.shape[0] + pr[:, 1]
        assert (pr[:, 0] < pr[:, 1]).all() and (np.diff(key) > 0).all()
        ref = inputs.aabb_candidates(pos, tris, inflate)
        assert pr.shape == ref.shape and (pr == ref).all()
        assert pr.shape[0] > 100


def test_generator_classifier_matches_oracle(oracle_mod):
    """The generators' orientation classifier (workload shaping only) agrees with the oracle's
    Moeller predicate, and the degeneracy filter keeps |tc| >= 1e-6 * edge (north_star)."""
    from paper_2606_06511_b200 import inputs
    for pb in (inputs.config1_icospheres(subdiv=3), inputs.config4_sweep(n_tris=3000, n_pairs=20000)):
        r = oracle_mod.pairs(pb.pos, pb.tris, pb.pairs, want_J=False)
        hit, deg = inputs.classify_pairs(pb.pos, pb.tris, pb.pairs)
        assert not deg.any()
        assert (hit == r["active"].astype(bool)).all()
        act = r["active"].astype(bool)
        P = pb.pos[pb.tris[pb.pairs[act]]]                                  # [A,2,3,3]
        e = np.linalg.norm(P - np.roll(P, 1, axis=2), axis=-1).mean(axis=(1, 2))
        assert (np.abs(r["tc"][act]).min(axis=1) >= 1e-6 * e).all()
    pb = inputs.config4_sweep(n_tris=3000, n_pairs=20000)
    assert abs(oracle_mod.pairs(pb.pos, pb.tris, pb.pairs, want_J=False)["active"].mean() - 0.5) < 0.01
