"""Parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times (config 4:
2 M-triangle soup, 10 M candidate pairs, ~50 % active; same generator, same seed, same three
C-ABI calls per step).

The oracle cannot assemble 10 M pairs in seconds, so the comparison is split the way the task
allows: what the oracle can compute pair by pair is compared on ALL pairs (active set bit-exact,
tc, per-pair energy, total energy); gradient, BSR rows and H.p are compared on SAMPLED vertices --
row v of the assembled Hessian only receives contributions from pairs that contain a triangle
owning v, so the oracle assembles exactly those pairs and its row v must equal the GPU's row v of
the full matrix (pattern bit-exact, values to tolerance).  Properties that hold at any size
(grad.x = 4E, sum of the gradient = 0, rowptr monotone, columns strictly ascending) close the rest.
"""
import numpy as np
import pytest
import torch

from helpers import mean_edge, rel, unpack_mask

pytestmark = pytest.mark.gpu

N_TRIS = 2_000_000
N_PAIRS = 10_000_000
CHUNK = 1_000_000
N_SAMPLE_TRIS = 400


def oracle_all_pairs(oracle, pos, tris, pairs, hess_mode, eps=1e-6):
    """Per-pair oracle results on ALL pairs (chunked: J is needed only for the FILTER margin and is
    dropped chunk by chunk).  Returns active, tc, T and the margin mask (True = keep)."""
    P = pairs.shape[0]
    active = np.zeros(P, dtype=bool)
    tc = np.zeros((P, 2))
    T = np.zeros(P)
    keep = np.ones(P, dtype=bool)
    for lo in range(0, P, CHUNK):
        hi = min(P, lo + CHUNK)
        r = oracle.pairs(pos, tris, pairs[lo:hi], 1.0, want_J=True)
        act = r["active"].astype(bool)
        e = mean_edge(pos, tris, pairs[lo:hi])
        bad = act & (np.abs(r["tc"]).min(axis=1) < eps * e)
        if hess_mode == 1:
            g0, g1 = r["J"][:, 0], r["J"][:, 1]
            d = np.abs((g0 * g1).sum(1))
            bad |= act & (d < eps * np.linalg.norm(g0, axis=1) * np.linalg.norm(g1, axis=1))
        active[lo:hi] = act
        tc[lo:hi] = r["tc"]
        T[lo:hi] = r["T"]
        keep[lo:hi] = ~bad
    return active, tc, T, keep


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_config4_full_size(oracle_mod, dtype):
    from paper_2606_06511_b200 import inputs, tt
    oracle = oracle_mod
    dev = torch.device("cuda:0")
    hess_mode = 1
    tdt = torch.float64 if dtype == "f64" else torch.float32
    tol = dict(e=1e-10, g=1e-10, h=1e-9, y=1e-9) if dtype == "f64" else dict(e=1e-4, g=1e-4, h=1e-3, y=1e-3)
    pb = inputs.config4_sweep(n_tris=N_TRIS, n_pairs=N_PAIRS, seed=inputs.BASE_SEED + 4, device="cuda:0")
    pos_np = pb.pos.astype(np.float32).astype(np.float64) if dtype == "f32" else pb.pos   # reading A12
    act_ref, tc_ref, T_ref, keep = oracle_all_pairs(oracle, pos_np, pb.tris, pb.pairs, hess_mode)
    pairs_np = np.ascontiguousarray(pb.pairs[keep])
    act_ref, tc_ref, T_ref = act_ref[keep], tc_ref[keep], T_ref[keep]
    P = pairs_np.shape[0]
    assert P > 0.99 * N_PAIRS * 0.99
    nV = pos_np.shape[0]

    ctx = tt.Context(tdt, hess_mode, 1.0, 0)
    pos = torch.from_numpy(pos_np).to(dev).to(tdt).contiguous()
    tris = torch.from_numpy(pb.tris).to(dev)
    prs = torch.from_numpy(pairs_np).to(dev)
    prob = ctx.problem(pos, tris, prs)

    # ---- a1 / a2 on ALL pairs: active set bit-exact, tc, per-pair and total energy ----
    e_sum = torch.zeros(1, dtype=tdt, device=dev)
    e_pp = torch.zeros(P, dtype=tdt, device=dev)
    mask = torch.zeros((P + 31) // 32, dtype=torch.int32, device=dev)
    tc = torch.zeros((P, 2), dtype=tdt, device=dev)
    na = torch.zeros(1, dtype=torch.int64, device=dev)
    ctx.tt_energy(prob, e_sum, e_pp, mask, tc, na)
    torch.cuda.synchronize()
    act = unpack_mask(mask.cpu().numpy().view(np.uint32), P)
    assert (act == act_ref).all(), "active set differs at %s" % np.nonzero(act != act_ref)[0][:10]
    assert int(na.cpu()[0]) == int(act_ref.sum())
    E_ref = float(np.sum(T_ref))            # pairwise (numpy) summation of the oracle's per-pair energies
    assert rel(e_sum.cpu().numpy()[0], E_ref) <= tol["e"]
    assert rel(e_pp.cpu().numpy(), T_ref) <= tol["e"]
    tcg = tc.cpu().numpy().astype(np.float64)
    assert np.abs(tcg - tc_ref).max() <= (1e-9 if dtype == "f64" else 1e-3) * np.abs(tc_ref).max()
    assert (tcg[~act_ref] == 0).all()
    del e_pp, tc, mask

    # ---- the step bench.py times: symbolic + numeric + H.p ----
    nnzb, n_active = ctx.tt_hess_symbolic(prob)
    assert n_active == int(act_ref.sum())
    energy = torch.zeros(1, dtype=tdt, device=dev)
    grad = torch.empty((nV, 3), dtype=tdt, device=dev)
    rowptr = torch.empty(nV + 1, dtype=torch.int32, device=dev)
    colind = torch.empty(nnzb, dtype=torch.int32, device=dev)
    vals = torch.empty((nnzb, 3, 3), dtype=tdt, device=dev)
    ctx.tt_energy_grad_hess(prob, energy, grad, rowptr, colind, vals, nnzb)
    p_np = np.random.default_rng(7).normal(size=(nV, 3))
    if dtype == "f32":
        p_np = p_np.astype(np.float32).astype(np.float64)
    pvec = torch.from_numpy(p_np).to(dev).to(tdt)
    y = torch.full_like(pvec, float("nan"))
    ctx.tt_hess_vec(prob, pvec, y)
    torch.cuda.synchronize()
    assert rel(energy.cpu().numpy()[0], E_ref) <= tol["e"]

    # ---- properties at full size ----
    rp = rowptr.cpu().numpy().astype(np.int64)
    assert rp[0] == 0 and rp[-1] == nnzb and (np.diff(rp) >= 0).all()
    ci_d = colind.to(torch.int64)
    row_of = torch.repeat_interleave(torch.arange(nV, device=dev), torch.from_numpy(np.diff(rp)).to(dev))
    key = row_of * nV + ci_d
    assert bool((key[1:] > key[:-1]).all()), "columns must be strictly ascending inside every row"
    del key, row_of, ci_d
    E = float(energy.cpu()[0])
    gx = float((grad.double() * pos.double()).sum().cpu())
    assert abs(gx - 4 * E) <= (1e-9 if dtype == "f64" else 1e-3) * 4 * E                      # I6
    assert float(grad.double().sum(0).abs().max().cpu()) <= (1e-9 if dtype == "f64" else 1e-3) * float(grad.abs().max().cpu()) * 100
    assert bool(torch.isfinite(y).all())

    # ---- sampled vertices: gradient, BSR rows, H.p against the oracle's assembly of the incident pairs ----
    rng = np.random.default_rng(11)
    touched = np.unique(pairs_np[act_ref].ravel())
    st = rng.choice(touched, size=N_SAMPLE_TRIS, replace=False)
    inc = np.isin(pairs_np[:, 0], st) | np.isin(pairs_np[:, 1], st)
    sub = np.ascontiguousarray(pairs_np[inc])
    ref = oracle.assemble(pos_np, pb.tris, sub, 1.0, hess_mode)
    rows = np.unique(pb.tris[st].ravel())
    g_gpu = grad[torch.from_numpy(rows).to(dev)].cpu().numpy().astype(np.float64)
    assert rel(g_gpu, ref["grad"][rows]) <= tol["g"]
    ci = colind.cpu().numpy()
    y_gpu = y.cpu().numpy().astype(np.float64)
    num = den = 0.0
    ynum = yden = 0.0
    n_blocks = 0
    for v in rows:
        a0, a1 = rp[v], rp[v + 1]
        b0, b1 = ref["rowptr"][v], ref["rowptr"][v + 1]
        assert a1 - a0 == b1 - b0 and a1 > a0, "row %d: %d blocks vs %d" % (v, a1 - a0, b1 - b0)
        assert (ci[a0:a1] == ref["colind"][b0:b1]).all()
        vg = vals[a0:a1].cpu().numpy().astype(np.float64)
        vr = ref["vals"][b0:b1].reshape(-1, 3, 3)
        num += ((vg - vr) ** 2).sum()
        den += (vr ** 2).sum()
        yr = np.einsum("bij,bj->i", vr, p_np[ref["colind"][b0:b1]])
        ynum += ((y_gpu[v] - yr) ** 2).sum()
        yden += (yr ** 2).sum()
        n_blocks += a1 - a0
    assert n_blocks > 10 * N_SAMPLE_TRIS
    assert np.sqrt(num / den) <= tol["h"]
    assert np.sqrt(ynum / yden) <= tol["y"]
    ctx.close()
