"""Seeded synthetic inputs shaped like BASELINE.json's five configs (recipe: DESIGN.md, "Inputs").

This module serves BOTH the CUDA path and the CPU oracle and therefore holds none of the
method's arithmetic: no Moeller intervals, no t_c, no energy, no derivatives.  What it does
hold is plain mesh construction, a broad-phase stand-in (inflated-AABB overlap on a uniform
grid -- the paper's spatial hash, is outside the hot path) and a textbook
orientation-determinant ("signed volume") classifier used only to shape the workload:
  * accept/reject random soup pairs to the requested intersecting fraction (config 4), and
  * drop near-degenerate pairs (a vertex within eps*edge of the other plane, two edge lines
    within eps*edge of each other, near-parallel planes), which keeps every discrete decision
    of the method -- and in particular |t_c^0|, |t_c^1| (BASELINE.json north_star) -- at least
    eps*edge away from flipping.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

BASE_SEED = 20260651  # seed of config i is BASE_SEED + i


@dataclass
class Problem:
    """pos [nV,3] float64, tris [nT,3] int32, pairs [P,2] int32 (triangle ids, candidates)."""
    pos: np.ndarray
    tris: np.ndarray
    pairs: np.ndarray
    name: str = ""
    meta: dict = field(default_factory=dict)

    @property
    def n_verts(self):
        return int(self.pos.shape[0])

    @property
    def n_tris(self):
        return int(self.tris.shape[0])

    @property
    def n_pairs(self):
        return int(self.pairs.shape[0])


# --------------------------------------------------------------------------------------------
# orientation determinants (textbook geometry; NOT the method)
# --------------------------------------------------------------------------------------------
class _NP:
    """numpy backend of the orientation classifier."""
    @staticmethod
    def asarray(a, like=None):
        return np.asarray(a)

    stack = staticmethod(lambda xs: np.stack(xs, axis=-1))
    norm = staticmethod(lambda a: np.linalg.norm(a, axis=-1))
    maximum = staticmethod(np.maximum)
    abs = staticmethod(np.abs)
    to_numpy = staticmethod(lambda a: np.asarray(a))

    @staticmethod
    def zeros_bool(n, like=None):
        return np.zeros(n, dtype=bool)


def _torch_backend(device):
    import torch

    class _TH:
        """torch backend (same arithmetic, any device) -- used by bench.py to shape 10M+ pair
        workloads in seconds on the GPU box; the pairs it keeps are then copied to the host."""
        @staticmethod
        def asarray(a, like=None):
            return torch.as_tensor(a, device=device)

        stack = staticmethod(lambda xs: torch.stack(xs, dim=-1))
        norm = staticmethod(lambda a: torch.linalg.norm(a, dim=-1))
        maximum = staticmethod(lambda a, b: torch.clamp(a, min=b))
        abs = staticmethod(torch.abs)
        to_numpy = staticmethod(lambda a: a.cpu().numpy())

        @staticmethod
        def zeros_bool(n, like=None):
            return torch.zeros(n, dtype=torch.bool, device=device)

    return _TH


def _cross(xp, a, b):
    return xp.stack([a[..., 1] * b[..., 2] - a[..., 2] * b[..., 1],
                     a[..., 2] * b[..., 0] - a[..., 0] * b[..., 2],
                     a[..., 0] * b[..., 1] - a[..., 1] * b[..., 0]])


def _dot(a, b):
    return (a * b).sum(-1)


def _orient(xp, p, q, r, s):
    """Signed volume (x6) of tetrahedron (p,q,r,s)."""
    return _dot(_cross(xp, q - p, r - p), s - p)


def _segment_pierces(xp, p, q, t0, t1, t2):
    """Closed segment pq crosses the interior of triangle (t0,t1,t2) (strict)."""
    dp = _orient(xp, t0, t1, t2, p)
    dq = _orient(xp, t0, t1, t2, q)
    s0 = _orient(xp, p, q, t0, t1)
    s1 = _orient(xp, p, q, t1, t2)
    s2 = _orient(xp, p, q, t2, t0)
    opposite = ((dp > 0) & (dq < 0)) | ((dp < 0) & (dq > 0))
    inside = ((s0 > 0) & (s1 > 0) & (s2 > 0)) | ((s0 < 0) & (s1 < 0) & (s2 < 0))
    return opposite & inside


def classify_pairs(pos, tris, pairs, eps=1e-6, chunk=1 << 20, device=None):
    """Returns (intersects[P] bool, degenerate[P] bool) from orientation determinants only.

    intersects: some edge of one triangle pierces the other (6 edge/triangle tests).
    degenerate: any vertex-plane distance, edge-line/edge-line distance or plane angle within
    eps (relative to the pair's mean edge length) of zero, or the pair shares a vertex index.
    device=None: numpy; otherwise a torch device string (same arithmetic in fp64).
    """
    xp = _NP if device is None else _torch_backend(device)
    P = pairs.shape[0]
    hit = np.zeros(P, dtype=bool)
    deg = np.zeros(P, dtype=bool)
    pos_x = xp.asarray(pos)
    tris_x = xp.asarray(tris if device is None else tris.astype(np.int64))
    tiny = float(np.finfo(np.float64).tiny)
    for lo in range(0, P, chunk):
        pr = xp.asarray(pairs[lo:lo + chunk] if device is None else pairs[lo:lo + chunk].astype(np.int64))
        ta = tris_x[pr[:, 0]]
        tb = tris_x[pr[:, 1]]
        A = pos_x[ta]  # [n,3,3]
        B = pos_x[tb]
        a = [A[:, 0], A[:, 1], A[:, 2]]
        b = [B[:, 0], B[:, 1], B[:, 2]]
        h = xp.zeros_bool(pr.shape[0])
        for i in range(3):
            h = h | _segment_pierces(xp, a[i], a[(i + 1) % 3], b[0], b[1], b[2])
            h = h | _segment_pierces(xp, b[i], b[(i + 1) % 3], a[0], a[1], a[2])
        # degeneracy measures
        ea = [a[1] - a[0], a[2] - a[1], a[0] - a[2]]
        eb = [b[1] - b[0], b[2] - b[1], b[0] - b[2]]
        L = sum(xp.norm(e) for e in ea + eb) / 6.0
        na = _cross(xp, a[1] - a[0], a[2] - a[0])
        nb = _cross(xp, b[1] - b[0], b[2] - b[0])
        lna = xp.norm(na)
        lnb = xp.norm(nb)
        d = (lna <= tiny) | (lnb <= tiny)
        lna = xp.maximum(lna, tiny)
        lnb = xp.maximum(lnb, tiny)
        for m in range(3):
            d = d | (xp.abs(_dot(nb, a[m] - b[0])) / lnb < eps * L)
            d = d | (xp.abs(_dot(na, b[m] - a[0])) / lna < eps * L)
        d = d | (xp.norm(_cross(xp, na, nb)) < eps * lna * lnb)
        for i in range(3):
            for j in range(3):
                c = _cross(xp, ea[i], eb[j])
                lc = xp.norm(c)
                lei = xp.norm(ea[i]) * xp.norm(eb[j])
                par = lc < eps * lei                       # near-parallel edges: no line distance
                dist = xp.abs(_dot(c, b[j] - a[i])) / xp.maximum(lc, tiny)
                d = d | ((~par) & (dist < eps * L))
        shared = (ta[:, :, None] == tb[:, None, :]).any(-1).any(-1)
        hit[lo:lo + chunk] = xp.to_numpy(h & ~shared)
        deg[lo:lo + chunk] = xp.to_numpy(d | shared)
    return hit, deg


def drop_adjacent(tris, pairs):
    """Remove candidate pairs whose triangles share a vertex index."""
    ta = tris[pairs[:, 0]]
    tb = tris[pairs[:, 1]]
    shared = (ta[:, :, None] == tb[:, None, :]).any(axis=(1, 2))
    return pairs[~shared]


def drop_degenerate(pos, tris, pairs, eps=1e-6):
    _, deg = classify_pairs(pos, tris, pairs, eps)
    return np.ascontiguousarray(pairs[~deg]), int(deg.sum())


# --------------------------------------------------------------------------------------------
# broad-phase stand-in: inflated-AABB overlap on a uniform grid
# --------------------------------------------------------------------------------------------
def aabb_candidates(pos, tris, inflate=0.0, max_pairs=None):
    """All pairs (i<j) of triangles whose AABBs, inflated by `inflate` on every side, overlap,
    with shared-vertex pairs dropped.  Sorted lexicographically.  Uniform-grid bucketing."""
    P = pos[tris]                                    # [nT,3,3]
    lo = P.min(axis=1) - inflate
    hi = P.max(axis=1) + inflate
    ext = (hi - lo).max()
    cell = float(ext) * 1.0001
    org = lo.min(axis=0)
    clo = np.floor((lo - org) / cell).astype(np.int64)
    chi = np.floor((hi - org) / cell).astype(np.int64)   # chi - clo in {0,1} per axis
    dims = chi.max(axis=0) + 1
    nT = tris.shape[0]
    ids, cells = [], []
    for dx in (0, 1):
        for dy in (0, 1):
            for dz in (0, 1):
                c = clo + np.array([dx, dy, dz])
                ok = (c <= chi).all(axis=1)
                t = np.nonzero(ok)[0]
                cc = c[ok]
                cells.append((cc[:, 0] * dims[1] + cc[:, 1]) * dims[2] + cc[:, 2])
                ids.append(t)
    ids = np.concatenate(ids)
    cells = np.concatenate(cells)
    order = np.lexsort((ids, cells))
    ids = ids[order]
    cells = cells[order]
    out = []
    n = ids.shape[0]
    d = 1
    total = 0
    while d < n:
        same = cells[:-d] == cells[d:]
        if not same.any():
            break
        i = ids[:-d][same]
        j = ids[d:][same]
        ov = ((lo[i] <= hi[j]) & (lo[j] <= hi[i])).all(axis=1)
        i, j = i[ov], j[ov]
        out.append(np.stack([np.minimum(i, j), np.maximum(i, j)], axis=1))
        total += i.shape[0]
        d += 1
    if not out:
        return np.zeros((0, 2), dtype=np.int32)
    pr = np.concatenate(out)
    key = np.unique(pr[:, 0] * np.int64(nT) + pr[:, 1])   # a pair can meet in several cells
    pr = np.stack([key // nT, key % nT], axis=1).astype(np.int32)
    pr = drop_adjacent(tris, pr)
    if max_pairs is not None and pr.shape[0] > max_pairs:
        pr = pr[:max_pairs]
    return np.ascontiguousarray(pr)


# --------------------------------------------------------------------------------------------
# meshes
# --------------------------------------------------------------------------------------------
def icosphere(subdiv):
    """Unit icosphere: 20*4^subdiv triangles."""
    t = (1.0 + np.sqrt(5.0)) / 2.0
    v = np.array([[-1, t, 0], [1, t, 0], [-1, -t, 0], [1, -t, 0], [0, -1, t], [0, 1, t],
                  [0, -1, -t], [0, 1, -t], [t, 0, -1], [t, 0, 1], [-t, 0, -1], [-t, 0, 1]], dtype=np.float64)
    v /= np.linalg.norm(v, axis=1, keepdims=True)
    f = np.array([[0, 11, 5], [0, 5, 1], [0, 1, 7], [0, 7, 10], [0, 10, 11], [1, 5, 9], [5, 11, 4],
                  [11, 10, 2], [10, 7, 6], [7, 1, 8], [3, 9, 4], [3, 4, 2], [3, 2, 6], [3, 6, 8],
                  [3, 8, 9], [4, 9, 5], [2, 4, 11], [6, 2, 10], [8, 6, 7], [9, 8, 1]], dtype=np.int64)
    for _ in range(subdiv):
        e = np.concatenate([f[:, [0, 1]], f[:, [1, 2]], f[:, [2, 0]]])
        e.sort(axis=1)
        ue, inv = np.unique(e, axis=0, return_inverse=True)
        inv = inv.reshape(-1)
        mid = v[ue[:, 0]] + v[ue[:, 1]]
        mid /= np.linalg.norm(mid, axis=1, keepdims=True)
        nv = v.shape[0]
        v = np.concatenate([v, mid])
        nf = f.shape[0]
        m01 = nv + inv[:nf]
        m12 = nv + inv[nf:2 * nf]
        m20 = nv + inv[2 * nf:]
        f = np.concatenate([np.stack([f[:, 0], m01, m20], 1), np.stack([f[:, 1], m12, m01], 1),
                            np.stack([f[:, 2], m20, m12], 1), np.stack([m01, m12, m20], 1)])
    return v, f.astype(np.int32)


def _grid_tris(nu, nv, wrap_u=False, wrap_v=False):
    """Two triangles per quad of an nu x nv vertex grid (periodic where asked)."""
    qu = nu if wrap_u else nu - 1
    qv = nv if wrap_v else nv - 1
    i, j = np.meshgrid(np.arange(qu), np.arange(qv), indexing="ij")
    i = i.reshape(-1)
    j = j.reshape(-1)
    i1 = (i + 1) % nu
    j1 = (j + 1) % nv
    v00 = i * nv + j
    v10 = i1 * nv + j
    v01 = i * nv + j1
    v11 = i1 * nv + j1
    t = np.concatenate([np.stack([v00, v10, v11], 1), np.stack([v00, v11, v01], 1)])
    return t.astype(np.int32)


def _finish(pos, tris, pairs, name, eps, meta):
    pairs, ndrop = drop_degenerate(pos, tris, pairs, eps) if eps else (pairs, 0)
    meta = dict(meta, dropped_degenerate=ndrop, eps=eps)
    return Problem(np.ascontiguousarray(pos, dtype=np.float64), np.ascontiguousarray(tris, dtype=np.int32),
                   np.ascontiguousarray(pairs, dtype=np.int32), name, meta)


# --------------------------------------------------------------------------------------------
# the five configs
# --------------------------------------------------------------------------------------------
def config0_soup(n_tris=64, seed=BASE_SEED + 0, eps=1e-6, pool=None):
    """Triangle soup, vertices uniform in [0,1]^3; candidates = all pairs, shared-vertex dropped.
    pool=None: every triangle owns its 3 vertices.  pool=k: indices drawn from k shared vertices
    (exercises the adjacency rule)."""
    rng = np.random.default_rng(seed)
    if pool is None:
        pos = rng.random((3 * n_tris, 3))
        tris = np.arange(3 * n_tris, dtype=np.int32).reshape(-1, 3)
    else:
        pos = rng.random((pool, 3))
        tris = np.stack([rng.permutation(pool)[:3] for _ in range(n_tris)]).astype(np.int32)
    i, j = np.triu_indices(n_tris, 1)
    pairs = drop_adjacent(tris, np.stack([i, j], 1).astype(np.int32))
    return _finish(pos, tris, pairs, "soup%d" % n_tris, eps, dict(seed=seed, pool=pool))


def config1_icospheres(subdiv=4, seed=BASE_SEED + 1, sep=0.6, jitter=1e-3, inflate=0.02, eps=1e-6):
    """Two unit icospheres, centres `sep` apart, vertex jitter N(0, jitter); inflated-AABB candidates."""
    rng = np.random.default_rng(seed)
    v, f = icosphere(subdiv)
    pos = np.concatenate([v, v + np.array([sep, 0.0, 0.0])])
    pos = pos + rng.normal(0.0, jitter, pos.shape)
    tris = np.concatenate([f, f + v.shape[0]]).astype(np.int32)
    pairs = aabb_candidates(pos, tris, inflate)
    return _finish(pos, tris, pairs, "icospheres%d" % subdiv, eps, dict(seed=seed, inflate=inflate))


def config2_cloth(n=256, seed=BASE_SEED + 2, jitter=1e-3, inflate=0.002, eps=1e-6):
    """n x n sheet, z = 0.3 sin(6 pi x) sin(4 pi y), mirror-folded about the middle vertex column
    (x' = x_h - |x - x_h|) so the two layers pass through each other; jitter N(0, jitter)."""
    rng = np.random.default_rng(seed)
    u = np.arange(n) / (n - 1.0)
    X, Y = np.meshgrid(u, u, indexing="ij")
    Z = 0.3 * np.sin(6 * np.pi * X) * np.sin(4 * np.pi * Y)
    xh = (n // 2) / (n - 1.0)
    Xf = xh - np.abs(X - xh)
    pos = np.stack([Xf, Y, Z], -1).reshape(-1, 3) + rng.normal(0.0, jitter, (n * n, 3))
    tris = _grid_tris(n, n)
    pairs = aabb_candidates(pos, tris, inflate)
    return _finish(pos, tris, pairs, "cloth%d" % n, eps, dict(seed=seed, inflate=inflate))


def config3_torus(nu=1000, nv=500, seed=BASE_SEED + 3, R=1.0, r=0.3, amp=0.25, inflate=0.0, eps=1e-6):
    """Torus (2*nu*nv triangles) with a seeded low-frequency twist + displacement field that
    pushes the tube through itself."""
    rng = np.random.default_rng(seed)
    th = 2 * np.pi * np.arange(nu) / nu
    ph = 2 * np.pi * np.arange(nv) / nv
    TH, PH = np.meshgrid(th, ph, indexing="ij")
    twist = 1.5 * np.sin(rng.integers(1, 4) * TH + rng.uniform(0, 2 * np.pi))   # twist of the tube angle
    PHt = PH + twist
    x = (R + r * np.cos(PHt)) * np.cos(TH)
    y = (R + r * np.cos(PHt)) * np.sin(TH)
    z = r * np.sin(PHt)
    pos = np.stack([x, y, z], -1).reshape(-1, 3)
    # Smooth displacement field of SPACE, d(x) = sum_m A_m sin(k_m.x + phi_m), with |A||k| > 1:
    # x -> x + d(x) is then not injective, so the tube folds through itself (a bijective
    # deformation such as a pure twist could never create a self-intersection).
    disp = np.zeros_like(pos)
    for _ in range(3):
        k = rng.normal(size=3)
        k *= (2 * np.pi * rng.uniform(1.0, 2.0)) / np.linalg.norm(k)
        A = rng.normal(size=3)
        A *= amp / np.linalg.norm(A)
        disp += A[None, :] * np.sin(pos @ k + rng.uniform(0, 2 * np.pi))[:, None]
    pos = pos + disp
    pos = pos + rng.normal(0.0, 1e-2 * (2 * np.pi * r / nv), pos.shape)
    tris = _grid_tris(nu, nv, wrap_u=True, wrap_v=True)
    pairs = aabb_candidates(pos, tris, inflate)
    return _finish(pos, tris, pairs, "torus%dx%d" % (nu, nv), eps, dict(seed=seed, inflate=inflate))


def config4_sweep(n_tris=2_000_000, n_pairs=10_000_000, seed=BASE_SEED + 4, frac_active=0.5, eps=1e-6,
                  device=None):
    """Random soup (own vertices, uniform [0,1]^3) with seeded random distinct non-adjacent
    candidate pairs, accepted/rejected with the orientation classifier to `frac_active`
    intersecting (the raw rate for uniform triangles is ~27.6 %).  Pair order is random.
    device: None = numpy classifier; a torch device string runs the same classifier there."""
    rng = np.random.default_rng(seed)
    pos = rng.random((3 * n_tris, 3))
    tris = np.arange(3 * n_tris, dtype=np.int32).reshape(-1, 3)
    want_hit = int(round(n_pairs * frac_active))
    want_miss = n_pairs - want_hit
    hits, misses = [], []
    nh = nm = 0
    seen_draws = 0
    while nh < want_hit or nm < want_miss:
        n = max(1 << 16, min(1 << 22, int(1.3 * max((want_hit - nh) / 0.27, (want_miss - nm) / 0.72))))
        i = rng.integers(0, n_tris, n, dtype=np.int64)
        j = rng.integers(0, n_tris, n, dtype=np.int64)
        ok = i != j
        pr = np.stack([i[ok], j[ok]], 1).astype(np.int32)
        h, d = classify_pairs(pos, tris, pr, eps, device=device)
        good = ~d
        ph = pr[good & h][:max(0, want_hit - nh)]
        pm = pr[good & ~h][:max(0, want_miss - nm)]
        hits.append(ph)
        misses.append(pm)
        nh += ph.shape[0]
        nm += pm.shape[0]
        seen_draws += n
    pairs = np.concatenate(hits + misses)
    # distinct pairs (unordered); duplicates are vanishingly rare but legal to drop
    key = np.minimum(pairs[:, 0], pairs[:, 1]).astype(np.int64) * n_tris + np.maximum(pairs[:, 0], pairs[:, 1])
    _, first = np.unique(key, return_index=True)
    pairs = pairs[np.sort(first)]
    pairs = pairs[rng.permutation(pairs.shape[0])]
    return Problem(pos, tris, np.ascontiguousarray(pairs, dtype=np.int32), "sweep%dk" % (n_pairs // 1000),
                   dict(seed=seed, eps=eps, draws=seen_draws, frac_active=frac_active))


def by_name(name, **kw):
    table = dict(config0=config0_soup, config1=config1_icospheres, config2=config2_cloth,
                 config3=config3_torus, config4=config4_sweep)
    return table[name](**kw)
