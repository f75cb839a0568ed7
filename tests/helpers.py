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
