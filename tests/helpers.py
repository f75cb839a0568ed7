"""Shared test helpers: oracle-side margin filter and GPU-vs-oracle comparison (tests only)."""
import numpy as np


def mean_edge(pos, tris, pairs):
    P = pos[tris[pairs]]                                   # [n,2,3,3]
    return np.linalg.norm(P - np.roll(P, 1, axis=2), axis=-1).mean(axis=(1, 2))


def filter_margins(oracle, pb, hess_mode, sigma=1.0, eps=1e-6):
    """BASELINE.json north_star: reject pairs with |tc0| or |tc1| below eps*edge.  The generators
    already keep every orientation determinant eps away from zero; this applies the literal
    criterion with the ORACLE's tc, plus (FILTER mode) the sign margin of g0.g1 (DESIGN.md G-margins)."""
    pairs = pb.pairs
    for _ in range(3):
        r = oracle.pairs(pb.pos, pb.tris, pairs, sigma, want_J=True)
        act = r["active"].astype(bool)
        bad = np.zeros(pairs.shape[0], dtype=bool)
        e = mean_edge(pb.pos, pb.tris, pairs)
        bad |= act & (np.abs(r["tc"]).min(axis=1) < eps * sigma * e)
        if hess_mode == 1:
            g0, g1 = r["J"][:, 0], r["J"][:, 1]
            d = np.abs((g0 * g1).sum(1))
            bad |= act & (d < eps * np.linalg.norm(g0, axis=1) * np.linalg.norm(g1, axis=1))
        if not bad.any():
            return pairs
        pairs = np.ascontiguousarray(pairs[~bad])
    return pairs


def rel(a, b):
    a = np.asarray(a, dtype=np.float64)
    b = np.asarray(b, dtype=np.float64)
    n = np.linalg.norm(b.ravel())
    d = np.linalg.norm((a - b).ravel())
    return d / n if n > 0 else d


def unpack_mask(mask_words, P):
    bits = np.unpackbits(mask_words.view(np.uint8), bitorder="little")
    return bits[:P].astype(bool)


# ---- per-row / per-block comparisons (VERDICT r1 "norm-only comparisons") ---------------------------
# A single global L2 / Frobenius norm cannot see one wrong small row or block inside a large result.
# These checks normalise every row / block by ITS OWN scale.  Bounds ("Tolerances"):
#   gradient row v : |dg_v| / sum_pairs |contribution of the pair to v|        <= ROW_TOL[dtype]["g"]
#   Hessian block  : |dH_pq|_F / (|H_pq|_F + 1e-3 |row p|_F)                   <= ROW_TOL[dtype]["h"]
#   H.p row v      : |dy_v| / sum_q |H_vq|_F |p_q|                             <= ROW_TOL[dtype]["y"]
# The denominators are sums of magnitudes, so cancellation inside a row cannot hide an error and a
# row whose contributions are 1e6 times below the largest row is still checked to the same relative bound.
ROW_TOL = {"f64": dict(g=1e-8, h=1e-7, y=1e-7), "f32": dict(g=2e-3, h=2e-2, y=2e-2)}


def grad_row_scale(nV, tris, pairs, ref):
    """sum over active pairs of |cg0 g0_v| + |cg1 g1_v| per vertex v (Eq. 3 magnitudes, from the
    oracle's J and tc; used only as a per-row error scale)."""
    act = ref["active"].astype(bool)
    tc = ref["tc"][act]
    J = ref["J"][act]                                      # [A,2,18]
    cg0 = np.abs(2.0 * tc[:, 0] * tc[:, 1] ** 2)
    cg1 = np.abs(2.0 * tc[:, 1] * tc[:, 0] ** 2)
    g0 = np.linalg.norm(J[:, 0].reshape(-1, 6, 3), axis=2)  # [A,6]
    g1 = np.linalg.norm(J[:, 1].reshape(-1, 6, 3), axis=2)
    contrib = cg0[:, None] * g0 + cg1[:, None] * g1
    verts = np.concatenate([tris[pairs[act, 0]], tris[pairs[act, 1]]], axis=1)   # [A,6]
    scale = np.zeros(nV)
    np.add.at(scale, verts.ravel(), contrib.ravel())
    return scale


def max_row_err(a, b, scale, rows=None):
    """max over rows (with scale > 0) of |a_v - b_v| / scale_v; rows without contributions must be exactly zero."""
    a = np.asarray(a, dtype=np.float64)
    b = np.asarray(b, dtype=np.float64)
    if rows is not None:
        a, b, scale = a[rows], b[rows], scale[rows]
    d = np.linalg.norm(a - b, axis=1)
    pos = scale > 0
    assert not a[~pos].any(), "rows no active pair touches must be exactly zero"
    return float((d[pos] / scale[pos]).max()) if pos.any() else 0.0


def max_block_err(vals, vals_ref, rowptr):
    """max over blocks of |dH_pq|_F / (|H_pq|_F + 1e-3 |row p|_F), same pattern on both sides."""
    v = np.asarray(vals, dtype=np.float64).reshape(-1, 9)
    r = np.asarray(vals_ref, dtype=np.float64).reshape(-1, 9)
    if r.shape[0] == 0:
        return 0.0
    num = np.linalg.norm(v - r, axis=1)
    bn = np.linalg.norm(r, axis=1)
    rp = np.asarray(rowptr, dtype=np.int64)
    row_of = np.repeat(np.arange(rp.shape[0] - 1), np.diff(rp))
    rown = np.sqrt(np.bincount(row_of, weights=bn ** 2, minlength=rp.shape[0] - 1))
    den = bn + 1e-3 * rown[row_of]
    ok = den > 0
    assert not v[~ok].any()
    return float((num[ok] / den[ok]).max())


def hp_row_scale(rowptr, colind, vals_ref, p):
    """sum_q |H_vq|_F |p_q| per row v."""
    r = np.asarray(vals_ref, dtype=np.float64).reshape(-1, 9)
    rp = np.asarray(rowptr, dtype=np.int64)
    nV = rp.shape[0] - 1
    if r.shape[0] == 0:
        return np.zeros(nV)
    row_of = np.repeat(np.arange(nV), np.diff(rp))
    w = np.linalg.norm(r, axis=1) * np.linalg.norm(np.asarray(p, dtype=np.float64)[colind], axis=1)
    return np.bincount(row_of, weights=w, minlength=nV)
