"""CPU oracle of the membrane term of the untangling demo -- TEST INFRASTRUCTURE, NOT THE PRODUCT (same rules as
oracle/__init__.py).

PAPER.md L41-43 (Fig. 2) optimises meshes from an invalid to a valid state inside a simulation whose elastic model it
does not give; SURVEY.md 8(f) NEXT-4 asks for the demo "with a simple membrane energy".  DESIGN.md reading A18 fixes the
simplest textbook one, an edge-spring (mass-spring) membrane on the mesh's own edges:

    E_m(x) = k/2  sum over the mesh's unique edges (i, j) of  (|x_i - x_j| - L_ij)^2,      L_ij = |r_i - r_j| at the rest positions r,

    grad_i  = k sum_j (|d| - L) d / |d|,                          d = x_i - x_j,
    H p     = sum over edges of  K (p_i - p_j)  at i  and  -K (p_i - p_j)  at j,
    K       = k [ n n^T + max(0, 1 - L / |d|) (I - n n^T) ],       n = d / |d|,

K is the edge's exact Hessian block with its negative (compressed-spring) part clamped to zero, the usual positive
semi-definite choice for Newton-type solvers; stretched edges have it exact.  Everything below is plain dense numpy in
fp64, written from these formulas; the consumer loop with the membrane (newton_step) follows oracle/newton.py step by
step with  E = E_T + E_m,  g = g_T + g_m,  H = H_T + H_m,  and a block-Jacobi preconditioner made of the MEMBRANE's
diagonal blocks plus mu I (the solve is matrix-free on the GPU, so the intersection Hessian's diagonal is not at hand).
"""
from __future__ import annotations

import numpy as np

from . import HESS_PSD2, assemble, broad_phase, pairs as _pairs


def edges_of(tris) -> np.ndarray:
    """Unique undirected edges (i < j) of a triangle list, sorted lexicographically."""
    t = np.asarray(tris, dtype=np.int64)
    e = np.concatenate([t[:, [0, 1]], t[:, [1, 2]], t[:, [2, 0]]])
    e = e[e[:, 0] != e[:, 1]]
    e.sort(axis=1)
    return np.unique(e, axis=0)


def energy_grad(pos, rest, tris, k: float):
    pos = np.asarray(pos, dtype=np.float64)
    rest = np.asarray(rest, dtype=np.float64)
    E = edges_of(tris)
    d = pos[E[:, 0]] - pos[E[:, 1]]
    ln = np.linalg.norm(d, axis=1)
    L = np.linalg.norm(rest[E[:, 0]] - rest[E[:, 1]], axis=1)
    energy = 0.5 * k * float(np.sum((ln - L) ** 2))
    f = (k * (ln - L) / ln)[:, None] * d
    g = np.zeros_like(pos)
    np.add.at(g, E[:, 0], f)
    np.add.at(g, E[:, 1], -f)
    return energy, g


def edge_blocks(pos, rest, tris, k: float):
    """The clamped 3x3 stiffness block K of every edge."""
    pos = np.asarray(pos, dtype=np.float64)
    rest = np.asarray(rest, dtype=np.float64)
    E = edges_of(tris)
    d = pos[E[:, 0]] - pos[E[:, 1]]
    ln = np.linalg.norm(d, axis=1)
    L = np.linalg.norm(rest[E[:, 0]] - rest[E[:, 1]], axis=1)
    n = d / ln[:, None]
    nn = n[:, :, None] * n[:, None, :]
    c = np.maximum(0.0, 1.0 - L / ln)
    K = k * (nn + c[:, None, None] * (np.eye(3)[None] - nn))
    return E, K


def hess_vec(pos, rest, tris, k: float, p):
    E, K = edge_blocks(pos, rest, tris, k)
    p = np.asarray(p, dtype=np.float64)
    dp = p[E[:, 0]] - p[E[:, 1]]
    f = np.einsum("eij,ej->ei", K, dp)
    y = np.zeros_like(p)
    np.add.at(y, E[:, 0], f)
    np.add.at(y, E[:, 1], -f)
    return y


def diag_blocks(pos, rest, tris, k: float):
    """Diagonal 3x3 blocks of the membrane Hessian: the sum of the K of a vertex's edges."""
    E, K = edge_blocks(pos, rest, tris, k)
    D = np.zeros((np.asarray(pos).shape[0], 3, 3))
    np.add.at(D, E[:, 0], K)
    np.add.at(D, E[:, 1], K)
    return D


def dense_hessian(pos, rest, tris, k: float):
    E, K = edge_blocks(pos, rest, tris, k)
    n = np.asarray(pos).shape[0]
    H = np.zeros((3 * n, 3 * n))
    for (i, j), Kb in zip(E, K):
        H[3 * i:3 * i + 3, 3 * i:3 * i + 3] += Kb
        H[3 * j:3 * j + 3, 3 * j:3 * j + 3] += Kb
        H[3 * i:3 * i + 3, 3 * j:3 * j + 3] -= Kb
        H[3 * j:3 * j + 3, 3 * i:3 * i + 3] -= Kb
    return H


def _bsr_dense(r, nV):
    H = np.zeros((3 * nV, 3 * nV))
    for v in range(nV):
        for e in range(r["rowptr"][v], r["rowptr"][v + 1]):
            c = r["colind"][e]
            H[3 * v:3 * v + 3, 3 * c:3 * c + 3] = r["vals"][e]
    return H


def pcg_dense(H, minv, b, max_iter: int):
    """Textbook preconditioned CG (the recurrences of oracle.pcg) on a dense operator, exactly max_iter steps from 0."""
    n = b.shape[0]
    x = np.zeros(n)
    r = b.copy()
    apply = lambda v: np.einsum("vij,vj->vi", minv, v.reshape(-1, 3)).ravel()
    z = apply(r)
    p = z.copy()
    rz = float(r @ z)
    for _ in range(max_iter):
        q = H @ p
        alpha = rz / float(p @ q)
        x += alpha * p
        r -= alpha * q
        z = apply(r)
        rz_new = float(r @ z)
        p = z + (rz_new / rz) * p
        rz = rz_new
    return x


def total_energy(pos, rest, tris, pair_ids, k: float, sigma: float = 1.0) -> float:
    return float(_pairs(pos, tris, pair_ids, sigma, want_J=False)["energy"]) + energy_grad(pos, rest, tris, k)[0]


def newton_step(pos, rest, tris, pair_ids, k: float, hess_mode: int = HESS_PSD2, mu: float = 1e-3, pcg_iter: int = 10,
                c1: float = 1e-4, max_backtrack: int = 20, sigma: float = 1.0) -> dict:
    """oracle/newton.py's step with E = E_T + E_m (small inputs: dense operator)."""
    pos = np.ascontiguousarray(pos, dtype=np.float64)
    nV = pos.shape[0]
    r = assemble(pos, tris, pair_ids, sigma, hess_mode)
    Em, gm = energy_grad(pos, rest, tris, k)
    E0 = float(r["energy"]) + Em
    g = r["grad"] + gm
    H = _bsr_dense(r, nV) + dense_hessian(pos, rest, tris, k) + mu * np.eye(3 * nV)
    minv = np.linalg.inv(diag_blocks(pos, rest, tris, k) + mu * np.eye(3)[None])
    d = pcg_dense(H, minv, g.ravel(), pcg_iter).reshape(nV, 3)
    gd = float(np.sum(g * d))
    out = dict(x=pos.copy(), E0=E0, E1=E0, gnorm=float(np.linalg.norm(g)), gd=gd, alpha=0.0, backtracks=0, accepted=False,
               n_active=int(r["active"].sum()), d=d, E_membrane=Em)
    if out["n_active"] == 0:        # reading A16: the loop's goal is "no pair is active"; nothing to do
        out.update(accepted=True, d=np.zeros_like(pos), gd=0.0)
        return out
    alpha = 1.0
    for j in range(max_backtrack + 1):
        x_try = pos - alpha * d
        E_try = total_energy(x_try, rest, tris, pair_ids, k, sigma)
        if E_try <= E0 - c1 * alpha * gd:
            out.update(x=x_try, E1=E_try, alpha=alpha, backtracks=j, accepted=True)
            return out
        alpha *= 0.5
    out["backtracks"] = max_backtrack + 1
    return out


def untangle(pos, rest, tris, k: float, inflate: float = 0.0, max_steps: int = 20, **kw) -> dict:
    """oracle/newton.py's untangle with the membrane term in every step."""
    x = np.ascontiguousarray(pos, dtype=np.float64).copy()
    hist = []
    for _ in range(max_steps):
        cand = broad_phase(x, tris, inflate)
        s = newton_step(x, rest, tris, cand, k, **kw)
        hist.append(dict(E0=s["E0"], E1=s["E1"], alpha=s["alpha"], n_active=s["n_active"], n_pairs=int(cand.shape[0]),
                         accepted=s["accepted"], x0=x, x1=s["x"]))
        if s["n_active"] == 0 or not s["accepted"]:
            break
        x = s["x"]
    return dict(x=x, history=hist)
