"""Parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times (same generator,
same seed, same three C-ABI calls per step):

  config 4 (throughput sweep)  2 M-triangle soup, 10 M candidate pairs, fp64 and fp32   (bench.py's default line)
  config 4 at the top of the sweep: 50 M pairs, fp64  (29 % of the triangles have more than 32 partners;
                                 value offsets pass 2^31)
  config 3 (twisted torus)     1000 x 500 quads = 1 M triangles, ~8.1 M candidates, fp64 and fp32
                                 (shared vertices: the general-row merge path at scale)

The oracle cannot assemble these sizes in seconds, so the comparison is split the way the task
allows: what the oracle can compute pair by pair is compared on ALL pairs (active set bit-exact,
tc, per-pair energy, total energy); gradient, BSR rows and H.p are compared on SAMPLED vertices --
row v of the assembled Hessian only receives contributions from pairs that contain a triangle
owning v, so the oracle assembles exactly those pairs and its row v must equal the GPU's row v of
the full matrix (pattern bit-exact, values to tolerance, globally AND per row / per block).
Properties that hold at any size (grad.x = 4E, sum of the gradient = 0, rowptr monotone, columns
strictly ascending) close the rest.
"""
import numpy as np
import pytest
import torch

from helpers import ROW_TOL, grad_row_scale, hp_row_scale, max_block_err, max_row_err, mean_edge, rel, unpack_mask

pytestmark = [pytest.mark.gpu, pytest.mark.slow]

N_TRIS = 2_000_000
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


def full_size_case(oracle, pb, dtype, hess_mode=1, n_sample=N_SAMPLE_TRIS, min_keep=0.98):
    from paper_2606_06511_b200 import tt
    dev = torch.device("cuda:0")
    tdt = torch.float64 if dtype == "f64" else torch.float32
    tol = dict(e=1e-10, g=1e-10, h=1e-9, y=1e-9) if dtype == "f64" else dict(e=1e-4, g=1e-4, h=1e-3, y=1e-3)
    rt = ROW_TOL[dtype]
    pos_np = pb.pos.astype(np.float32).astype(np.float64) if dtype == "f32" else pb.pos   # reading A12
    act_ref, tc_ref, T_ref, keep = oracle_all_pairs(oracle, pos_np, pb.tris, pb.pairs, hess_mode)
    pairs_np = np.ascontiguousarray(pb.pairs[keep])
    act_ref, tc_ref, T_ref = act_ref[keep], tc_ref[keep], T_ref[keep]
    P = pairs_np.shape[0]
    assert P > min_keep * pb.n_pairs
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
    epp = e_pp.cpu().numpy().astype(np.float64)
    assert rel(epp, T_ref) <= tol["e"]
    # per pair, each against its own value (not only the global norm)
    assert (np.abs(epp - T_ref)[act_ref] / T_ref[act_ref]).max() <= (1e-7 if dtype == "f64" else 1e-5)
    tcg = tc.cpu().numpy().astype(np.float64)
    assert np.abs(tcg - tc_ref).max() <= (1e-9 if dtype == "f64" else 1e-3) * np.abs(tc_ref).max()
    assert (tcg[~act_ref] == 0).all() and (epp[~act_ref] == 0).all()
    del e_pp, tc, mask, epp, tcg

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
    assert bool(torch.isfinite(y).all()) and bool(torch.isfinite(vals).all())

    # ---- sampled vertices: gradient, BSR rows, H.p against the oracle's assembly of the incident pairs ----
    rng = np.random.default_rng(11)
    touched = np.unique(pairs_np[act_ref].ravel())
    st = rng.choice(touched, size=min(n_sample, touched.shape[0]), replace=False)
    rows = np.unique(pb.tris[st].ravel())
    tri_set = np.nonzero(np.isin(pb.tris, rows).any(axis=1))[0]      # every triangle that owns a sampled vertex
    inc = np.isin(pairs_np[:, 0], tri_set) | np.isin(pairs_np[:, 1], tri_set)
    sub = np.ascontiguousarray(pairs_np[inc])
    ref = oracle.assemble(pos_np, pb.tris, sub, 1.0, hess_mode)
    g_full = grad.cpu().numpy().astype(np.float64)
    assert rel(g_full[rows], ref["grad"][rows]) <= tol["g"]
    assert max_row_err(g_full, ref["grad"], grad_row_scale(nV, pb.tris, sub, ref), rows) <= rt["g"]
    ci = colind.cpu().numpy()
    y_gpu = y.cpu().numpy().astype(np.float64)
    vg_all, vr_all, rp_loc, y_ref_rows, y_scale = [], [], [0], [], []
    for v in rows:
        a0, a1 = rp[v], rp[v + 1]
        b0, b1 = ref["rowptr"][v], ref["rowptr"][v + 1]
        assert a1 - a0 == b1 - b0 and a1 > a0, "row %d: %d blocks vs %d" % (v, a1 - a0, b1 - b0)
        assert (ci[a0:a1] == ref["colind"][b0:b1]).all()
        vg_all.append(vals[a0:a1].cpu().numpy().astype(np.float64))
        vr = ref["vals"][b0:b1].reshape(-1, 3, 3)
        vr_all.append(vr)
        rp_loc.append(rp_loc[-1] + (a1 - a0))
        pc = p_np[ref["colind"][b0:b1]]
        y_ref_rows.append(np.einsum("bij,bj->i", vr, pc))
        y_scale.append((np.linalg.norm(vr.reshape(-1, 9), axis=1) * np.linalg.norm(pc, axis=1)).sum())
    vg_all, vr_all = np.concatenate(vg_all), np.concatenate(vr_all)
    assert vg_all.shape[0] > 10 * rows.shape[0] / 3
    assert rel(vg_all, vr_all) <= tol["h"]
    assert max_block_err(vg_all, vr_all, np.asarray(rp_loc)) <= rt["h"]
    y_ref_rows = np.asarray(y_ref_rows)
    assert rel(y_gpu[rows], y_ref_rows) <= tol["y"]
    assert max_row_err(y_gpu[rows], y_ref_rows, np.asarray(y_scale)) <= rt["y"]
    stats = ctx.tt_stats()
    ctx.close()
    return stats, dict(P=P, n_active=n_active, nnzb=nnzb)


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_config4_full_size(oracle_mod, dtype):
    """bench.py's default line: 10 M pairs."""
    from paper_2606_06511_b200 import inputs
    pb = inputs.config4_sweep(n_tris=N_TRIS, n_pairs=10_000_000, seed=inputs.BASE_SEED + 4, device="cuda:0")
    st, sz = full_size_case(oracle_mod, pb, dtype)
    assert st["blocks_merged"] == 0


def test_config4_top_of_sweep_50M(oracle_mod):
    """BASELINE.json configs[4] "1M-50M": the 50 M point, fp64.  The value count nnzb * 9 exceeds 2^31 (33.7 GB of blocks) and about 29 % of
    the touched triangles have more than 32 partners (the long-triangle paths of K4 and K6)."""
    from paper_2606_06511_b200 import inputs
    pb = inputs.config4_sweep(n_tris=N_TRIS, n_pairs=50_000_000, seed=inputs.BASE_SEED + 4, device="cuda:0")
    st, sz = full_size_case(oracle_mod, pb, "f64")
    assert sz["nnzb"] * 9 > 2 ** 31          # value offsets do not fit an int32
    deg = np.bincount(pb.pairs.ravel(), minlength=N_TRIS)           # candidates per triangle (~2x the active degree)
    assert (deg > 64).mean() > 0.05
    # triangles with more than 32 ACTIVE partners: split into parts (soup: always splittable) or rounds of their own
    assert st["split_triangles"] + st["long_rounds"] > 0.05 * st["n_touched_tris"]


_torus = {}


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_config3_full_size(oracle_mod, dtype):
    """BASELINE.json configs[3] at its stated size: 1 M triangles, ~8.1 M candidates, Hessian assembled to BSR,
    fp64 and fp32.  Shared vertices: every row goes through the general-row merge (record sort, k_merge)."""
    from paper_2606_06511_b200 import inputs
    if "pb" not in _torus:
        _torus["pb"] = inputs.config3_torus()
    pb = _torus["pb"]
    assert pb.n_tris == 1_000_000 and pb.n_pairs > 7_000_000
    st, sz = full_size_case(oracle_mod, pb, dtype, n_sample=400, min_keep=0.99)
    assert st["blocks_merged"] > 0 and sz["n_active"] > 10_000
