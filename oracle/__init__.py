"""CPU oracle for arXiv 2606.06511 -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Thin ctypes wrapper over ``oracle/tt_oracle.cpp`` (plain fp64 C++, forward-mode dual numbers,
App. A of PAPER.md step by step).  Only ``tests/``, ``__graft_entry__.smoke()`` and the
``cpu_baseline`` / ``--impl reference`` legs of ``bench.py`` may import this package; the CUDA
product path (``paper_2606_06511_b200``) never does and shares no code with it.

Argument marshalling only -- every arithmetic step lives in the C++ file, next to the PAPER.md
line it follows.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "tt_oracle.cpp"
_LIB = _HERE / "libtt_oracle.so"

HESS_EQ4, HESS_FILTER, HESS_PSD2, HESS_PSDPROJ, HESS_EXACT = 0, 1, 2, 3, 4

_lib = None


def build(force: bool = False) -> Path:
    """Compile the oracle (g++ -O2 -ffp-contract=off -fopenmp).  Idempotent."""
    if force or not _LIB.exists() or _LIB.stat().st_mtime < _SRC.stat().st_mtime:
        cmd = ["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC",
               str(_SRC), "-o", str(_LIB)]
        subprocess.run(cmd, check=True)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        build()
        lib = ctypes.CDLL(str(_LIB))
        c_dp = ctypes.POINTER(ctypes.c_double)
        c_ip = ctypes.POINTER(ctypes.c_int32)
        c_bp = ctypes.POINTER(ctypes.c_uint8)
        i64 = ctypes.c_int64
        lib.tt_oracle_pair.argtypes = [c_dp, ctypes.c_double, ctypes.c_int, ctypes.POINTER(ctypes.c_int),
                                       c_dp, c_dp, c_dp, c_dp, c_dp, c_dp, c_dp]
        lib.tt_oracle_pair.restype = None
        lib.tt_oracle_pairs.argtypes = [c_dp, i64, c_ip, i64, c_ip, i64, ctypes.c_double, c_bp, c_dp,
                                        c_dp, c_dp, ctypes.c_int]
        lib.tt_oracle_pairs.restype = ctypes.c_double
        lib.tt_oracle_bsr_pattern.argtypes = [i64, c_ip, c_ip, i64, c_bp, c_ip, c_ip]
        lib.tt_oracle_bsr_pattern.restype = i64
        lib.tt_oracle_assemble.argtypes = [i64, c_ip, c_ip, i64, c_bp, c_dp, c_dp, ctypes.c_int, c_ip,
                                           c_ip, c_dp, c_dp]
        lib.tt_oracle_assemble.restype = None
        lib.tt_oracle_hess_vec_pairs.argtypes = [i64, c_ip, c_ip, i64, c_bp, c_dp, c_dp, ctypes.c_int,
                                                 c_dp, c_dp]
        lib.tt_oracle_hess_vec_pairs.restype = None
        lib.tt_oracle_bsr_matvec.argtypes = [i64, c_ip, c_ip, c_dp, c_dp, c_dp]
        lib.tt_oracle_bsr_matvec.restype = None
        lib.tt_oracle_broad_phase.argtypes = [c_dp, c_ip, i64, ctypes.c_double, c_ip, i64]
        lib.tt_oracle_broad_phase.restype = i64
        lib.tt_oracle_pair_exact.argtypes = [c_dp, ctypes.c_double, ctypes.POINTER(ctypes.c_int), c_dp, c_dp, c_dp, c_dp,
                                             c_dp, c_dp]
        lib.tt_oracle_pair_exact.restype = None
        lib.tt_oracle_exact_hess_vec.argtypes = [c_dp, i64, c_ip, c_ip, i64, ctypes.c_double, c_dp, c_dp]
        lib.tt_oracle_exact_hess_vec.restype = None
        lib.tt_oracle_assemble_exact.argtypes = [c_dp, i64, c_ip, c_ip, i64, c_bp, ctypes.c_double, c_ip, c_ip, c_dp]
        lib.tt_oracle_assemble_exact.restype = None
        lib.tt_oracle_block_jacobi.argtypes = [i64, c_ip, c_ip, c_dp, ctypes.c_double, c_dp]
        lib.tt_oracle_block_jacobi.restype = None
        lib.tt_oracle_pcg.argtypes = [i64, c_ip, c_ip, c_dp, ctypes.c_double, c_dp, c_dp, i64, ctypes.c_double,
                                      c_dp, c_dp, c_dp]
        lib.tt_oracle_pcg.restype = i64
        lib.tt_oracle_max_threads.argtypes = []
        lib.tt_oracle_max_threads.restype = ctypes.c_int
        _lib = lib
    return _lib


def _dp(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double)) if a is not None else None


def _ip(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_int32)) if a is not None else None


def _bp(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_uint8)) if a is not None else None


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _i32(a):
    return np.ascontiguousarray(a, dtype=np.int32)


def max_threads() -> int:
    return int(_load().tt_oracle_max_threads())


def pair(x, sigma: float = 1.0, hess_mode: int = HESS_FILTER) -> dict:
    """One pair, x = [a0,a1,a2,b0,b1,b2] (18 doubles).  Returns every per-pair quantity."""
    lib = _load()
    x = _f64(x).reshape(18)
    active = ctypes.c_int(0)
    tc = np.zeros(2)
    T = np.zeros(1)
    g0 = np.zeros(18)
    g1 = np.zeros(18)
    grad = np.zeros(18)
    H = np.zeros((18, 18))
    lam = np.zeros(3)
    lib.tt_oracle_pair(_dp(x), float(sigma), int(hess_mode), ctypes.byref(active), _dp(tc), _dp(T),
                       _dp(g0), _dp(g1), _dp(grad), _dp(H), _dp(lam))
    return dict(active=bool(active.value), tc=tc, energy=float(T[0]), g0=g0, g1=g1, grad=grad, H=H,
                lam=lam)


def pairs(pos, tris, pair_ids, sigma: float = 1.0, want_J: bool = True, n_threads: int = 0) -> dict:
    """Steps 1-9 for every candidate: active flags, tc, per-pair energy, J=[g0;g1], energy sum."""
    lib = _load()
    pos = _f64(pos)
    tris = _i32(tris)
    pair_ids = _i32(pair_ids).reshape(-1, 2)
    P = pair_ids.shape[0]
    active = np.zeros(P, dtype=np.uint8)
    tc = np.zeros((P, 2))
    T = np.zeros(P)
    J = np.zeros((P, 2, 18)) if want_J else None
    E = lib.tt_oracle_pairs(_dp(pos), pos.shape[0], _ip(tris), tris.shape[0], _ip(pair_ids), P,
                            float(sigma), _bp(active), _dp(tc), _dp(T), _dp(J), int(n_threads))
    return dict(energy=float(E), active=active, tc=tc, T=T, J=J)


def assemble(pos, tris, pair_ids, sigma: float = 1.0, hess_mode: int = HESS_FILTER,
             want_hess: bool = True, n_threads: int = 0) -> dict:
    """Whole hot path: energy, gradient [nV,3], BSR (rowptr, colind, vals[nnzb,3,3])."""
    lib = _load()
    pos = _f64(pos)
    tris = _i32(tris)
    pair_ids = _i32(pair_ids).reshape(-1, 2)
    nV, P = pos.shape[0], pair_ids.shape[0]
    r = pairs(pos, tris, pair_ids, sigma, True, n_threads)
    rowptr = np.zeros(nV + 1, dtype=np.int32)
    out = dict(r)
    grad = np.zeros((nV, 3))
    if want_hess:
        nnzb = lib.tt_oracle_bsr_pattern(nV, _ip(tris), _ip(pair_ids), P, _bp(r["active"]), _ip(rowptr),
                                         None)
        colind = np.zeros(max(int(nnzb), 1), dtype=np.int32)
        lib.tt_oracle_bsr_pattern(nV, _ip(tris), _ip(pair_ids), P, _bp(r["active"]), _ip(rowptr),
                                  _ip(colind))
        vals = np.zeros((max(int(nnzb), 1), 3, 3))
        lib.tt_oracle_assemble(nV, _ip(tris), _ip(pair_ids), P, _bp(r["active"]), _dp(r["tc"]),
                               _dp(r["J"]), HESS_EQ4 if hess_mode == HESS_EXACT else int(hess_mode), _ip(rowptr), _ip(colind),
                               _dp(grad), _dp(vals))
        if hess_mode == HESS_EXACT:   # same pattern, same gradient; the values from second-order duals
            lib.tt_oracle_assemble_exact(_dp(pos), nV, _ip(tris), _ip(pair_ids), P, _bp(r["active"]), float(sigma),
                                         _ip(rowptr), _ip(colind), _dp(vals))
        out.update(rowptr=rowptr, colind=colind[:nnzb], vals=vals[:nnzb], nnzb=int(nnzb))
    else:
        lib.tt_oracle_assemble(nV, _ip(tris), _ip(pair_ids), P, _bp(r["active"]), _dp(r["tc"]),
                               _dp(r["J"]), int(hess_mode), _ip(rowptr), None, _dp(grad), None)
    out["grad"] = grad
    return out


def hess_vec_pairs(nV, tris, pair_ids, active, tc, J, p, hess_mode: int = HESS_FILTER):
    """H.p as the sum over active pairs of J^T M (J p_loc)."""
    lib = _load()
    tris = _i32(tris)
    pair_ids = _i32(pair_ids).reshape(-1, 2)
    p = _f64(p)
    y = np.zeros((nV, 3))
    lib.tt_oracle_hess_vec_pairs(nV, _ip(tris), _ip(pair_ids), pair_ids.shape[0],
                                 _bp(np.ascontiguousarray(active, dtype=np.uint8)), _dp(_f64(tc)),
                                 _dp(_f64(J)), int(hess_mode), _dp(p), _dp(y))
    return y


def broad_phase(pos, tris, inflate: float = 0.0):
    """All non-adjacent triangle pairs i < j whose inflated AABBs overlap, lexicographic, by testing
    every pair.  Returns int32 [n,2]."""
    lib = _load()
    pos = _f64(pos)
    tris = _i32(tris)
    n = lib.tt_oracle_broad_phase(_dp(pos), _ip(tris), tris.shape[0], float(inflate), None, 0)
    out = np.zeros((max(int(n), 1), 2), dtype=np.int32)
    lib.tt_oracle_broad_phase(_dp(pos), _ip(tris), tris.shape[0], float(inflate), _ip(out), int(n))
    return out[:int(n)]


def bsr_matvec(rowptr, colind, vals, p):
    """Plain BSR(3x3) times vector."""
    lib = _load()
    rowptr = _i32(rowptr)
    nV = rowptr.shape[0] - 1
    p = _f64(p)
    y = np.zeros((nV, 3))
    colind = _i32(colind) if len(colind) else np.zeros(1, dtype=np.int32)
    vals = _f64(vals) if len(vals) else np.zeros((1, 3, 3))
    lib.tt_oracle_bsr_matvec(nV, _ip(rowptr), _ip(colind), _dp(vals), _dp(p), _dp(y))
    return y


def block_jacobi(rowptr, colind, vals, shift: float = 0.0):
    """Inverses of the 3x3 diagonal blocks of (H + shift I): [nV,3,3]."""
    lib = _load()
    rowptr = _i32(rowptr)
    nV = rowptr.shape[0] - 1
    colind = _i32(colind) if len(colind) else np.zeros(1, dtype=np.int32)
    vals = _f64(vals) if len(vals) else np.zeros((1, 3, 3))
    minv = np.zeros((nV, 3, 3))
    lib.tt_oracle_block_jacobi(nV, _ip(rowptr), _ip(colind), _dp(vals), float(shift), _dp(minv))
    return minv


def pcg(rowptr, colind, vals, b, shift: float = 0.0, max_iter: int = 50, rtol: float = 0.0, precond: bool = True,
        history: bool = False) -> dict:
    """Textbook preconditioned CG for (H + shift I) x = b from x_0 = 0, block-Jacobi preconditioner
    (precond=False: plain CG).  Returns x, iters, res (|r_k| per step) and, with history, every iterate."""
    lib = _load()
    rowptr = _i32(rowptr)
    nV = rowptr.shape[0] - 1
    colind = _i32(colind) if len(colind) else np.zeros(1, dtype=np.int32)
    vals = _f64(vals) if len(vals) else np.zeros((1, 3, 3))
    b = _f64(b).reshape(nV, 3)
    minv = block_jacobi(rowptr, colind, vals, shift) if precond else None
    x = np.zeros((nV, 3))
    xh = np.zeros((max_iter + 1, nV, 3)) if history else None
    res = np.zeros(max_iter + 1)
    k = lib.tt_oracle_pcg(nV, _ip(rowptr), _ip(colind), _dp(vals), float(shift), _dp(minv), _dp(b), int(max_iter),
                          float(rtol), _dp(x), _dp(xh), _dp(res))
    k = int(k)
    return dict(x=x, iters=k, res=res[:k + 1], x_hist=None if xh is None else xh[:k + 1], minv=minv)


def pair_exact(x, sigma: float = 1.0) -> dict:
    """One pair in second-order duals: the EXACT Hessian of T = (tc0 tc1)^2 (second half)
    plus the second derivatives H0, H1 of tc0, tc1."""
    lib = _load()
    x = _f64(x).reshape(18)
    active = ctypes.c_int(0)
    tc, T, grad = np.zeros(2), np.zeros(1), np.zeros(18)
    H, H0, H1 = np.zeros((18, 18)), np.zeros((18, 18)), np.zeros((18, 18))
    lib.tt_oracle_pair_exact(_dp(x), float(sigma), ctypes.byref(active), _dp(tc), _dp(T), _dp(grad), _dp(H), _dp(H0),
                             _dp(H1))
    return dict(active=bool(active.value), tc=tc, energy=float(T[0]), grad=grad, H=H, H0=H0, H1=H1)


def exact_hess_vec(pos, tris, pair_ids, p, sigma: float = 1.0):
    """y = H_exact p over all active pairs."""
    lib = _load()
    pos = _f64(pos)
    tris = _i32(tris)
    pair_ids = _i32(pair_ids).reshape(-1, 2)
    p = _f64(p)
    y = np.zeros_like(pos)
    lib.tt_oracle_exact_hess_vec(_dp(pos), pos.shape[0], _ip(tris), _ip(pair_ids), pair_ids.shape[0], float(sigma),
                                 _dp(p), _dp(y))
    return y
