"""CPU oracle of the consumer loop -- TEST INFRASTRUCTURE, NOT THE PRODUCT (same rules as oracle/__init__.py).

PAPER.md L5 names "a GPU-based inexact Newton optimization route" and L41-43 (Fig. 2) show meshes being untangled by
it; neither gives a formula, a tolerance or a step rule (SURVEY.md 8(f) NEXT-2 "line search on tt_energy ... all
choices would be ours", NEXT-4).  The operation is therefore its textbook definition (Nocedal & Wright, Alg. 3.1 +
7.1: line-search Newton-CG with a Levenberg-Marquardt shift), written out step by step on the oracle's routines, in
fp64 numpy.  DESIGN.md reading A16 fixes every choice:

  one step, for a FIXED candidate list:
    E0, g, H      = energy (Eq. 2), gradient (Eq. 3) and Hessian (Eq. 4 in the given hess_mode) at x
    d             = k-step block-Jacobi PCG approximation of (H + mu I)^-1 g from 0      (inexact Newton: truncated)
    alpha         = first of 1, 1/2, 1/4, ... (at most max_backtrack halvings) with
                    E(x - alpha d) <= E0 - c1 alpha g.d                                  (Armijo)
    x_new         = x - alpha d            (x unchanged if no alpha is accepted)
  untangle: repeat { candidates = broad phase at x (inflated AABBs); one step } until no pair is active.
"""
from __future__ import annotations

import numpy as np

from . import HESS_PSD2, assemble, broad_phase, pairs as _pairs, pcg


def energy(pos, tris, pair_ids, sigma: float = 1.0) -> float:
    """E = sum of T over the candidate list (Eq. 2)."""
    return float(_pairs(pos, tris, pair_ids, sigma, want_J=False)["energy"])


def newton_step(pos, tris, pair_ids, hess_mode: int = HESS_PSD2, mu: float = 1e-3, pcg_iter: int = 20,
                pcg_rtol: float = 0.0, c1: float = 1e-4, max_backtrack: int = 20, sigma: float = 1.0) -> dict:
    pos = np.ascontiguousarray(pos, dtype=np.float64)
    r = assemble(pos, tris, pair_ids, sigma, hess_mode)
    E0, g = float(r["energy"]), r["grad"]
    n_active = int(r["active"].sum())
    out = dict(x=pos.copy(), E0=E0, E1=E0, gnorm=float(np.linalg.norm(g)), gd=0.0, alpha=0.0, backtracks=0,
               accepted=False, n_active=n_active, pcg_iters=0, d=np.zeros_like(pos))
    if n_active == 0:
        out["accepted"] = True       # nothing intersects: x is a minimiser (E = 0)
        return out
    sol = pcg(r["rowptr"], r["colind"], r["vals"], g, shift=mu, max_iter=pcg_iter, rtol=pcg_rtol, precond=True)
    d = sol["x"]
    gd = float(np.sum(g * d))
    out.update(d=d, gd=gd, pcg_iters=int(sol["iters"]))
    alpha = 1.0
    for j in range(max_backtrack + 1):
        x_try = pos - alpha * d
        E_try = energy(x_try, tris, pair_ids, sigma)
        if E_try <= E0 - c1 * alpha * gd:
            out.update(x=x_try, E1=E_try, alpha=alpha, backtracks=j, accepted=True)
            return out
        alpha *= 0.5
    out["backtracks"] = max_backtrack + 1
    return out


def untangle(pos, tris, inflate: float = 0.0, max_steps: int = 20, **kw) -> dict:
    x = np.ascontiguousarray(pos, dtype=np.float64).copy()
    hist = []
    for _ in range(max_steps):
        cand = broad_phase(x, tris, inflate)
        s = newton_step(x, tris, cand, **kw)
        hist.append(dict(E0=s["E0"], E1=s["E1"], alpha=s["alpha"], n_active=s["n_active"], n_pairs=int(cand.shape[0]),
                         accepted=s["accepted"], x0=x, x1=s["x"]))
        if s["n_active"] == 0 or not s["accepted"]:
            break
        x = s["x"]
    return dict(x=x, history=hist)
