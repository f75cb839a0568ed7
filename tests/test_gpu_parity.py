"""GPU parity (-m gpu): the CUDA path, called through the C ABI, against the CPU oracle on the
same seeded inputs.  Bars (BASELINE.json north_star, A13): active set bit-exact;
fp64 energy/gradient rel 1e-10, Hessian blocks Frobenius-rel 1e-9 (pattern exact), H.p rel 1e-9;
fp32 variant 1e-4 / 1e-3."""
import numpy as np
import pytest

from helpers import (ROW_TOL, filter_margins, grad_row_scale, hp_row_scale, max_block_err, max_row_err, rel,
                     unpack_mask)

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

TOL = {"f64": dict(e=1e-10, g=1e-10, h=1e-9, y=1e-9, tc=1e-10),
       "f32": dict(e=1e-4, g=1e-4, h=1e-3, y=1e-3, tc=1e-4)}


def _dev():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    return torch.device("cuda:0")


def run_case(oracle, pb, dtype="f64", hess_mode=1, sigma=1.0, flags=0, check_vals=True, check_energy_call=True):
    from paper_2606_06511_b200 import tt
    dev = _dev()
    tdt = torch.float64 if dtype == "f64" else torch.float32
    pos_np = pb.pos.astype(np.float32).astype(np.float64) if dtype == "f32" else pb.pos   # A12
    pbo = type(pb)(pos_np, pb.tris, pb.pairs, pb.name, pb.meta)
    pairs = filter_margins(oracle, pbo, hess_mode, sigma)
    ref = oracle.assemble(pos_np, pb.tris, pairs, sigma, hess_mode)
    tol = TOL[dtype]
    ctx = tt.Context(tdt, hess_mode, sigma, 0, flags)
    pos = torch.from_numpy(pos_np).to(dev).to(tdt).contiguous()
    tris = torch.from_numpy(pb.tris).to(dev)
    prs = torch.from_numpy(pairs).to(dev)
    P = pairs.shape[0]
    act_ref = ref["active"].astype(bool)

    if check_energy_call:
        prob = ctx.problem(pos, tris, prs)
        e_sum = torch.zeros(1, dtype=tdt, device=dev)
        e_pp = torch.zeros(max(P, 1), dtype=tdt, device=dev)
        mask = torch.zeros(max((P + 31) // 32, 1), dtype=torch.int32, device=dev)
        tc = torch.zeros((max(P, 1), 2), dtype=tdt, device=dev)
        na = torch.zeros(1, dtype=torch.int64, device=dev)
        ctx.tt_energy(prob, e_sum, e_pp, mask, tc, na)
        torch.cuda.synchronize()
        act = unpack_mask(mask.cpu().numpy().view(np.uint32), P)
        assert (act == act_ref).all(), "active set differs at %s" % np.nonzero(act != act_ref)[0][:10]
        assert int(na.cpu()[0]) == int(act_ref.sum())
        assert rel(e_sum.cpu().numpy()[0], ref["energy"]) <= tol["e"]
        if P:
            tcg = tc.cpu().numpy().astype(np.float64)[:P]
            scale = np.abs(ref["tc"]).max() if act_ref.any() else 1.0
            assert np.abs(tcg - ref["tc"]).max() <= max(tol["tc"], 1e-12) * scale * 10
            assert (tcg[~act_ref] == 0).all()
            epp = e_pp.cpu().numpy().astype(np.float64)[:P]
            assert rel(epp, ref["T"]) <= tol["e"]

    out = tt.assemble(ctx, pos, tris, prs, want_hess=True)
    torch.cuda.synchronize()
    assert out["n_active"] == int(act_ref.sum())
    assert rel(out["energy"].cpu().numpy()[0], ref["energy"]) <= tol["e"]
    assert rel(out["grad"].cpu().numpy(), ref["grad"]) <= tol["g"]
    rt = ROW_TOL[dtype]
    nV = pos_np.shape[0]
    # every gradient row against ITS OWN contribution scale (a wrong small row cannot hide in the global norm)
    assert max_row_err(out["grad"].cpu().numpy(), ref["grad"], grad_row_scale(nV, pb.tris, pairs, ref)) <= rt["g"]
    assert out["nnzb"] == ref["nnzb"]
    assert (out["rowptr"].cpu().numpy() == ref["rowptr"]).all()
    assert (out["colind"].cpu().numpy() == ref["colind"]).all()
    if check_vals:
        assert rel(out["vals"].cpu().numpy(), ref["vals"]) <= tol["h"]
        # every block against its own norm (+ 1e-3 of its row's): one mis-scattered block fails here
        assert max_block_err(out["vals"].cpu().numpy(), ref["vals"], ref["rowptr"]) <= rt["h"]
    # gradient-only call must agree with the full call
    e2 = torch.zeros(1, dtype=tdt, device=dev)
    g2 = torch.empty_like(out["grad"])
    ctx.tt_energy_grad_hess(out["prob"], e2, g2)
    torch.cuda.synchronize()
    # (K6 sums a triangle's entries in a fixed shuffle-tree order, K4 sequentially: equal up to rounding order)
    assert rel(g2.cpu().numpy(), out["grad"].cpu().numpy()) <= (1e-13 if dtype == "f64" else 1e-6)
    assert rel(e2.cpu().numpy(), out["energy"].cpu().numpy()) <= (1e-14 if dtype == "f64" else 1e-6)
    # matrix-free H.p (a5) == oracle's per-pair J^T M J p == BSR.p (P10)
    rng = np.random.default_rng(12345)
    p_np = rng.normal(size=pos_np.shape)
    if dtype == "f32":
        p_np = p_np.astype(np.float32).astype(np.float64)
    p = torch.from_numpy(p_np).to(dev).to(tdt)
    y = torch.full_like(p, float("nan"))
    ctx.tt_hess_vec(out["prob"], p, y)
    torch.cuda.synchronize()
    if hess_mode == 4:   # exact Hessian: the oracle's second-order duals, pair by pair
        y_ref = oracle.exact_hess_vec(pos_np, pb.tris, pairs, p_np, sigma)
    else:
        y_ref = oracle.hess_vec_pairs(pos_np.shape[0], pb.tris, pairs, ref["active"], ref["tc"], ref["J"], p_np, hess_mode)
    assert rel(y.cpu().numpy(), y_ref) <= tol["y"]
    assert max_row_err(y.cpu().numpy(), y_ref, hp_row_scale(ref["rowptr"], ref["colind"], ref["vals"], p_np)) <= rt["y"]
    y_bsr = oracle.bsr_matvec(out["rowptr"].cpu().numpy(), out["colind"].cpu().numpy(),
                              out["vals"].cpu().numpy().astype(np.float64), p_np)
    assert rel(y_bsr, y_ref) <= tol["y"]
    stats = ctx.tt_stats()
    ctx.close()
    return ref, out, stats


# ------------------------------------------------------------------------------------ configs
@pytest.mark.parametrize("mode", [0, 1, 2, 3])
@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_config0_soup(oracle_mod, mode, dtype):
    from paper_2606_06511_b200 import inputs
    ref, out, st = run_case(oracle_mod, inputs.config0_soup(), dtype, mode)
    assert st["blocks_merged"] == 0          # own-vertex soup: every row is exclusive (long triangles included)
    assert 500 < out["n_active"] < 800


@pytest.mark.parametrize("flags", [0, 1])
def test_config0_shared_vertex_pool(oracle_mod, flags):
    """Triangles drawn from a small vertex pool: adjacency rule + general (merge) rows."""
    from paper_2606_06511_b200 import inputs
    pb = inputs.config0_soup(n_tris=64, pool=48, seed=77)
    ref, out, st = run_case(oracle_mod, pb, "f64", 1, flags=flags)
    assert st["blocks_merged"] > 0


def test_config0_forced_general_rows_equal_exclusive(oracle_mod):
    """TT_FLAG_FORCE_GENERAL_ROWS routes every row through the merge path: same matrix."""
    from paper_2606_06511_b200 import inputs
    pb = inputs.config0_soup()
    _, a, sa = run_case(oracle_mod, pb, "f64", 1, flags=0, check_energy_call=False)
    _, b, sb = run_case(oracle_mod, pb, "f64", 1, flags=1, check_energy_call=False)
    assert sa["blocks_merged"] == 0 and sb["blocks_direct"] == 0
    assert torch.equal(a["colind"], b["colind"]) and torch.equal(a["rowptr"], b["rowptr"])
    assert rel(a["vals"].cpu().numpy(), b["vals"].cpu().numpy()) < 1e-14


def test_psd_projection_mode_meshes(oracle_mod):
    """hess_mode 3 (PSD projection, closed 2x2 form on the GPU vs dense Jacobi in the oracle) on shared
    vertices (general rows) and on the icospheres; the assembled matrix is PSD on a small case."""
    from paper_2606_06511_b200 import inputs
    ref, out, st = run_case(oracle_mod, inputs.config0_soup(n_tris=48, pool=40, seed=5), "f64", 3)
    assert st["blocks_merged"] > 0
    run_case(oracle_mod, inputs.config1_icospheres(), "f64", 3)
    pb = inputs.config0_soup(n_tris=24, seed=9)
    ref, out, st = run_case(oracle_mod, pb, "f64", 3)
    nV = pb.n_verts
    H = np.zeros((3 * nV, 3 * nV))
    rp, ci, va = out["rowptr"].cpu().numpy(), out["colind"].cpu().numpy(), out["vals"].cpu().numpy()
    for r in range(nV):
        for e in range(rp[r], rp[r + 1]):
            H[3 * r:3 * r + 3, 3 * ci[e]:3 * ci[e] + 3] = va[e]
    w = np.linalg.eigvalsh(0.5 * (H + H.T))
    assert w[0] > -1e-9 * w[-1]
    assert np.abs(H - H.T).max() <= 1e-9 * np.abs(H).max()


def test_sigma_half(oracle_mod):
    from paper_2606_06511_b200 import inputs
    run_case(oracle_mod, inputs.config0_soup(), "f64", 0, sigma=0.5)


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_config1_icospheres(oracle_mod, dtype):
    from paper_2606_06511_b200 import inputs
    ref, out, st = run_case(oracle_mod, inputs.config1_icospheres(), dtype, 1)
    assert out["n_active"] > 100 and st["blocks_merged"] > 0


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_config2_cloth(oracle_mod, dtype):
    from paper_2606_06511_b200 import inputs
    ref, out, st = run_case(oracle_mod, inputs.config2_cloth(), dtype, 1)
    assert out["n_active"] > 1000


def test_config3_torus_reduced(oracle_mod):
    """Config 3's recipe at 1/25 of the triangles (full size: tests/test_gpu_full.py, slow)."""
    from paper_2606_06511_b200 import inputs
    run_case(oracle_mod, inputs.config3_torus(nu=200, nv=100), "f64", 1)
    run_case(oracle_mod, inputs.config3_torus(nu=200, nv=100), "f32", 1)


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_config4_sweep_reduced(oracle_mod, dtype):
    """Config 4's recipe, 60k triangles / 300k pairs: several CTA chunks, ragged tail, ~5 partners per triangle."""
    from paper_2606_06511_b200 import inputs
    pb = inputs.config4_sweep(n_tris=60_000, n_pairs=300_007)
    ref, out, st = run_case(oracle_mod, pb, dtype, 1)
    assert st["blocks_merged"] == 0
    assert abs(out["n_active"] / pb.n_pairs - 0.5) < 0.01


@pytest.mark.parametrize("n_tris,n_pairs,dtype", [(6000, 60_000, "f64"), (6000, 60_000, "f32"), (3000, 70_000, "f64")])
def test_bin_packed_segment_order(oracle_mod, n_tris, n_pairs, dtype):
    """10 and 23 partners per triangle on average: the entry segments are laid out in best-fit-decreasing order inside
    buckets of 128 triangles (k_bucket_order) and, in the second case, mixed with triangles that are split into parts; the
    matrix must not change (rows are addressed through rowbase) and the rounds must fill better than id order would."""
    from paper_2606_06511_b200 import inputs
    pb = inputs.config4_sweep(n_tris=n_tris, n_pairs=n_pairs, seed=777)
    ref, out, st = run_case(oracle_mod, pb, dtype, 1)
    assert st["blocks_merged"] == 0
    assert st["n_directed"] / (32.0 * st["rounds"]) > 0.9          # lane fill (id order: ~0.80 at these degrees)
    if n_tris == 3000:
        assert st["split_triangles"] > 50


@pytest.mark.parametrize("n_pairs,dtype", [(24_000, "f64"), (24_000, "f32"), (60_000, "f64")])
@pytest.mark.parametrize("layout", ["soup", "shuffled"])
def test_long_triangles(oracle_mod, n_pairs, dtype, layout):
    """Few triangles, many pairs each.  24k pairs: ~60 partners per triangle; 60k pairs: ~150.
    layout "soup" (vertex ids 3t, 3t+1, 3t+2): every triangle with more than 32 partners is SPLIT into parts
    that ride in ordinary rounds (k_long_prep, part slots in K4 / K6, k_split_finish).
    layout "shuffled" (the same soup with its vertex ids randomly permuted): the partners' columns interleave,
    so no long triangle can be split and all three long-triangle kernels run (k_assemble_long_tile<true> for
    33..64 partners, <false> for 65..127, k_assemble_long_direct beyond), rows still exclusive."""
    from paper_2606_06511_b200 import inputs
    pb = inputs.config4_sweep(n_tris=400, n_pairs=n_pairs, seed=4242)
    if layout == "shuffled":
        perm = np.random.default_rng(1).permutation(pb.n_verts)          # new id of old vertex v = perm[v]
        pos = np.empty_like(pb.pos)
        pos[perm] = pb.pos
        pb = inputs.Problem(pos, perm[pb.tris].astype(np.int32), pb.pairs, pb.name + "_shuffled", pb.meta)
    ref, out, st = run_case(oracle_mod, pb, dtype, 1)
    deg = np.bincount(pb.pairs[ref["active"].astype(bool)].ravel(), minlength=400)
    if n_pairs == 24_000:
        assert ((deg > 32) & (deg <= 64)).sum() > 50 and ((deg > 64) & (deg <= 127)).sum() > 30 and (deg <= 32).sum() > 20
    else:
        assert (deg > 127).sum() > 50
    assert st["blocks_merged"] == 0
    assert (st["split_triangles"] > 50) if layout == "soup" else (st["split_triangles"] == 0 and st["long_rounds"] > 50)


def test_long_triangles_shared_vertices(oracle_mod):
    """Long triangles on a shared-vertex pool: not splittable, general (merge) rows, all four hess modes' worth of
    structure in one: k_tri_symbolic ranking with duplicates, the long kernels writing to the merge workspace."""
    from paper_2606_06511_b200 import inputs
    pb = inputs.config0_soup(n_tris=260, pool=400, seed=31)
    ref, out, st = run_case(oracle_mod, pb, "f64", 1)
    deg = np.bincount(pb.pairs[ref["active"].astype(bool)].ravel(), minlength=260)
    assert (deg > 32).sum() > 20 and st["blocks_merged"] > 0 and st["long_rounds"] > 20


# ------------------------------------------------------------------------------------ edge cases
@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_vertex_exactly_on_plane(oracle_mod, dtype):
    """App. A L106-115 (reading A4): a vertex lying exactly on the other plane (+,-,0).  The recorded
    configuration marks that end-point as the vertex itself; all four placements (a or b carries the
    vertex, it is the smaller or the larger end-point) must match the oracle's one-sided derivative."""
    from paper_2606_06511_b200 import inputs
    a = np.array([[-1, -1, 0], [3, -1, 0], [1, 1, 0.0]])
    b = np.array([[0, 0, -1], [6, 0, 1], [1, 0, 0.0]])          # b2 on plane(a): tc = (-3, 1)
    mirror = np.array([-1.0, 1.0, 1.0])                         # x -> -x: vertex end-point becomes the larger one
    tris_pos, shift = [], np.array([10.0, 0, 0])
    for k, (ta, tb) in enumerate([(a, b), (b, a), (a * mirror, b * mirror), (b[[1, 2, 0]] * mirror, a[[2, 0, 1]] * mirror)]):
        tris_pos += [ta + k * shift, tb + k * shift]
    pos = np.concatenate(tris_pos)
    tris = np.arange(pos.shape[0], dtype=np.int32).reshape(-1, 3)
    pairs = np.array([[0, 1], [2, 3], [4, 5], [6, 7]], dtype=np.int32)
    pb = inputs.Problem(pos, tris, pairs, "on_plane", {})
    ref, out, st = run_case(oracle_mod, pb, dtype, 0)
    assert out["n_active"] == 4
    np.testing.assert_allclose(ref["tc"][0], [-3, 1], atol=1e-14)


def test_empty_and_inactive_inputs(oracle_mod):
    from paper_2606_06511_b200 import inputs, tt
    dev = _dev()
    pb = inputs.config0_soup()
    ctx = tt.Context(torch.float64, 1, 1.0, 0)
    pos = torch.from_numpy(pb.pos).to(dev)
    tris = torch.from_numpy(pb.tris).to(dev)
    # no candidates at all
    empty = torch.zeros((0, 2), dtype=torch.int32, device=dev)
    out = tt.assemble(ctx, pos, tris, empty)
    torch.cuda.synchronize()
    assert out["nnzb"] == 0 and out["n_active"] == 0
    assert float(out["energy"].cpu()[0]) == 0.0 and not out["grad"].cpu().numpy().any()
    assert not out["rowptr"].cpu().numpy().any()
    # candidates, none active (each triangle against a far-away copy)
    pos2 = torch.cat([pos, pos + 10.0])
    tris2 = torch.cat([tris, tris + pos.shape[0]])
    pairs2 = torch.stack([torch.arange(64), torch.arange(64) + 64], 1).to(torch.int32).to(dev)
    out = tt.assemble(ctx, pos2, tris2, pairs2)
    p = torch.randn_like(pos2)
    y = torch.full_like(p, float("nan"))
    ctx.tt_hess_vec(out["prob"], p, y)
    torch.cuda.synchronize()
    assert out["nnzb"] == 0 and out["n_active"] == 0 and not y.cpu().numpy().any()
    assert float(out["energy"].cpu()[0]) == 0.0 and not out["grad"].cpu().numpy().any()
    ctx.close()


def test_duplicate_and_reversed_candidates(oracle_mod):
    """The same pair listed twice and once reversed: legal input, contributions add up."""
    from paper_2606_06511_b200 import inputs
    pb = inputs.config0_soup()
    extra = np.concatenate([pb.pairs, pb.pairs[:300], pb.pairs[100:400, ::-1]])
    pb2 = type(pb)(pb.pos, pb.tris, np.ascontiguousarray(extra), "dups", {})
    run_case(oracle_mod, pb2, "f64", 1)


def test_error_paths(oracle_mod):
    from paper_2606_06511_b200 import inputs, tt
    dev = _dev()
    pb = inputs.config0_soup()
    ctx = tt.Context(torch.float64, 1, 1.0, 0)
    pos = torch.from_numpy(pb.pos).to(dev)
    tris = torch.from_numpy(pb.tris).to(dev)
    prs = torch.from_numpy(pb.pairs).to(dev)
    prob = ctx.problem(pos, tris, prs)
    e = torch.zeros(1, dtype=torch.float64, device=dev)
    g = torch.zeros_like(pos)
    with pytest.raises(tt.TTError) as ei:          # numeric before symbolic
        ctx.tt_energy_grad_hess(prob, e, g)
    assert ei.value.status == -5
    nnzb, _ = ctx.tt_hess_symbolic(prob)
    rp = torch.zeros(pos.shape[0] + 1, dtype=torch.int32, device=dev)
    ci = torch.zeros(nnzb, dtype=torch.int32, device=dev)
    va = torch.zeros((nnzb, 3, 3), dtype=torch.float64, device=dev)
    with pytest.raises(tt.TTError) as ei:          # capacity too small
        ctx.tt_energy_grad_hess(prob, e, g, rp, ci, va, nnzb - 1)
    assert ei.value.status == -4
    with pytest.raises(tt.TTError) as ei:          # aliased p / y
        ctx.tt_hess_vec(prob, g, g)
    assert ei.value.status == -1
    ctx.tt_energy_grad_hess(prob, e, g, rp, ci, va, nnzb)   # still usable after errors
    torch.cuda.synchronize()
    ctx.close()


def test_positions_moved_after_symbolic(oracle_mod):
    """K4 / K6 replay the branch decisions recorded by tt_hess_symbolic.  A Newton or
    line-search update of `pos` IN PLACE (same pointer) must not be evaluated with the stale decisions:
    tt_energy_grad_hess and tt_hess_vec return TT_ERR_STATE until tt_hess_symbolic is called again, and the
    result then equals the oracle at the NEW positions."""
    from paper_2606_06511_b200 import inputs, tt
    dev = _dev()
    pb = inputs.config0_soup()
    ctx = tt.Context(torch.float64, 1, 1.0, 0)
    pos = torch.from_numpy(pb.pos).to(dev)
    tris = torch.from_numpy(pb.tris).to(dev)
    prs = torch.from_numpy(pb.pairs).to(dev)
    prob = ctx.problem(pos, tris, prs)
    nnzb, _ = ctx.tt_hess_symbolic(prob)
    e = torch.zeros(1, dtype=torch.float64, device=dev)
    g = torch.zeros_like(pos)
    ctx.tt_energy_grad_hess(prob, e, g)                       # unchanged positions: fine
    saved = pos.clone()
    pos += 0.05 * torch.from_numpy(np.random.default_rng(3).normal(size=pb.pos.shape)).to(dev)   # in place
    with pytest.raises(tt.TTError) as ei:
        ctx.tt_energy_grad_hess(prob, e, g)
    assert ei.value.status == -5 and "positions changed" in str(ei.value)
    with pytest.raises(tt.TTError) as ei:
        ctx.tt_hess_vec(prob, g, torch.empty_like(g))
    assert ei.value.status == -5
    pos.copy_(saved)                                           # bit-identical positions again: accepted
    ctx.tt_energy_grad_hess(prob, e, g)
    pos[7, 2] += 1e-13                                         # one changed value (a few ulps) is enough
    with pytest.raises(tt.TTError):
        ctx.tt_energy_grad_hess(prob, e, g)
    # re-running the symbolic phase at the new positions gives the oracle's result there
    pos += 0.05 * torch.from_numpy(np.random.default_rng(4).normal(size=pb.pos.shape)).to(dev)
    pb2 = inputs.Problem(pos.cpu().numpy(), pb.tris, pb.pairs, "moved", {})
    pairs2 = filter_margins(oracle_mod, pb2, 1)
    ref = oracle_mod.assemble(pb2.pos, pb2.tris, pairs2, 1.0, 1)
    out = tt.assemble(ctx, pos, tris, torch.from_numpy(pairs2).to(dev))
    torch.cuda.synchronize()
    assert out["n_active"] == int(ref["active"].sum()) and out["nnzb"] == ref["nnzb"]
    assert rel(out["grad"].cpu().numpy(), ref["grad"]) <= 1e-10
    assert rel(out["vals"].cpu().numpy(), ref["vals"]) <= 1e-9
    # TT_FLAG_NO_STATE_CHECK: the caller vouches for the positions, no check is made
    ctx2 = tt.Context(torch.float64, 1, 1.0, 0, tt.TT_FLAG_NO_STATE_CHECK)
    prob2 = ctx2.problem(pos, tris, prs)
    ctx2.tt_hess_symbolic(prob2)
    pos[0, 0] += 1e-9
    ctx2.tt_energy_grad_hess(prob2, e, g)
    torch.cuda.synchronize()
    ctx.close()
    ctx2.close()


def test_validate_indices_flag(oracle_mod):
    """TT_FLAG_VALIDATE_INDICES: an out-of-range vertex or triangle index is reported, not dereferenced;
    valid input gives the same result as without the flag."""
    from paper_2606_06511_b200 import inputs, tt
    dev = _dev()
    pb = inputs.config0_soup()
    ctx = tt.Context(torch.float64, 1, 1.0, 0, tt.TT_FLAG_VALIDATE_INDICES)
    pos = torch.from_numpy(pb.pos).to(dev)
    tris = torch.from_numpy(pb.tris).to(dev)
    prs = torch.from_numpy(pb.pairs).to(dev)
    e = torch.zeros(1, dtype=torch.float64, device=dev)
    bad_tris = tris.clone()
    bad_tris[5, 1] = pos.shape[0]                       # one past the last vertex
    with pytest.raises(tt.TTError) as ei:
        ctx.tt_hess_symbolic(ctx.problem(pos, bad_tris, prs))
    assert ei.value.status == -1 and "1 vertex indices" in str(ei.value)
    bad_prs = prs.clone()
    bad_prs[7, 0] = -1
    bad_prs[9, 1] = tris.shape[0]
    with pytest.raises(tt.TTError) as ei:
        ctx.tt_energy(ctx.problem(pos, tris, bad_prs), e)
    assert ei.value.status == -1 and "2 triangle indices" in str(ei.value)
    with pytest.raises(tt.TTError):
        ctx.tt_broad_phase(pos, bad_tris, 0.0)
    out = tt.assemble(ctx, pos, tris, prs)             # valid input: unchanged behaviour
    ref = oracle_mod.assemble(pb.pos, pb.tris, pb.pairs, 1.0, 1)
    torch.cuda.synchronize()
    assert out["nnzb"] == ref["nnzb"] and out["n_active"] == int(ref["active"].sum())
    ctx.close()


def test_host_buffer_entry_point(oracle_mod):
    """tt_energy_grad_hess_host (the e2e call bench.py times) == device-buffer path == oracle."""
    from paper_2606_06511_b200 import inputs, tt
    _dev()
    pb = inputs.config4_sweep(n_tris=20_000, n_pairs=100_000)
    pairs = filter_margins(oracle_mod, pb, 1)
    ref = oracle_mod.assemble(pb.pos, pb.tris, pairs, 1.0, 1)
    ctx = tt.Context(torch.float64, 1, 1.0, 0)
    pos_h = torch.from_numpy(pb.pos).pin_memory()
    tris_h = torch.from_numpy(pb.tris).pin_memory()
    pairs_h = torch.from_numpy(pairs).pin_memory()
    e_h = torch.zeros(1, dtype=torch.float64).pin_memory()
    g_h = torch.zeros((pb.n_verts, 3), dtype=torch.float64).pin_memory()
    rp_h = torch.zeros(pb.n_verts + 1, dtype=torch.int32)
    cap = ref["nnzb"]
    ci_h = torch.zeros(cap, dtype=torch.int32)
    va_h = torch.zeros((cap, 3, 3), dtype=torch.float64)
    nnzb, na = ctx.tt_energy_grad_hess_host(pos_h, tris_h, pairs_h, e_h, g_h, rp_h, ci_h, va_h, cap)
    assert nnzb == ref["nnzb"] and na == int(ref["active"].sum())
    assert rel(e_h.numpy()[0], ref["energy"]) <= 1e-10
    assert rel(g_h.numpy(), ref["grad"]) <= 1e-10
    assert (rp_h.numpy() == ref["rowptr"]).all() and (ci_h.numpy() == ref["colind"]).all()
    assert rel(va_h.numpy(), ref["vals"]) <= 1e-9
    ctx.close()


def test_properties_on_gpu_outputs(oracle_mod):
    """Invariants that hold at any size, checked on the GPU's own outputs (config 4 recipe):
    grad.x = 4E, H_EQ4 x = 3 grad (I6), rows of H sum to zero against translations, symmetry."""
    from paper_2606_06511_b200 import inputs, tt
    dev = _dev()
    pb = inputs.config4_sweep(n_tris=50_000, n_pairs=250_000, seed=99)
    ctx = tt.Context(torch.float64, 0, 1.0, 0)
    pos = torch.from_numpy(pb.pos).to(dev)
    out = tt.assemble(ctx, pos, torch.from_numpy(pb.tris).to(dev), torch.from_numpy(pb.pairs).to(dev))
    y = torch.empty_like(pos)
    ctx.tt_hess_vec(out["prob"], pos, y)
    ones = torch.zeros_like(pos)
    ones[:, 1] = 1.0
    z = torch.empty_like(pos)
    ctx.tt_hess_vec(out["prob"], ones, z)
    torch.cuda.synchronize()
    E = float(out["energy"].cpu()[0])
    g = out["grad"]
    assert abs(float((g * pos).sum().cpu()) - 4 * E) <= 1e-9 * 4 * E
    assert float((y - 3 * g).norm().cpu()) <= 1e-9 * float((3 * g).norm().cpu())
    assert float(z.norm().cpu()) <= 1e-9 * float(out["vals"].norm().cpu())
    assert float(g.sum(0).abs().max().cpu()) <= 1e-9 * float(g.abs().max().cpu()) * 100
    ctx.close()


def test_hess_pattern_views(oracle_mod):
    """tt_hess_pattern: the ctx-owned pattern views equal the pattern tt_energy_grad_hess copies out, and a numeric call
    that is handed the views (no copy) writes the same values."""
    from paper_2606_06511_b200 import inputs, tt
    dev = _dev()
    pb = inputs.config0_soup(n_tris=64, pool=48, seed=77)
    ctx = tt.Context(torch.float64, 1, 1.0, 0)
    pos, tris, prs = (torch.from_numpy(a).to(dev) for a in (pb.pos, pb.tris, pb.pairs))
    out = tt.assemble(ctx, pos, tris, prs)
    rp, ci, nnzb = ctx.tt_hess_pattern(pb.n_verts)
    assert nnzb == out["nnzb"] and torch.equal(rp, out["rowptr"]) and torch.equal(ci[:nnzb], out["colind"])
    vals2 = torch.full_like(out["vals"], float("nan"))
    e2 = torch.zeros(1, dtype=torch.float64, device=dev)
    g2 = torch.empty_like(out["grad"])
    a_rp, a_ci, _ = ctx.tt_hess_pattern_ptrs()
    assert a_rp == rp.data_ptr() and a_ci == ci.data_ptr()
    ctx.tt_energy_grad_hess(out["prob"], e2, g2, a_rp, a_ci, vals2, nnzb)
    torch.cuda.synchronize()
    assert torch.equal(vals2, out["vals"]) and torch.equal(g2, out["grad"])
    ctx.close()
    ctx3 = tt.Context(torch.float64, 1, 1.0, 0)
    with pytest.raises(tt.TTError) as ei:
        ctx3.tt_hess_pattern_ptrs()
    assert ei.value.status == -5
    ctx3.close()


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_bit_reproducible_run_to_run(oracle_mod, dtype):
    """no floating-point atomics, every sum in a fixed order -- although the counting-sort scatter of K2 places
    entries with integer atomics, the segments are sorted before anything depends on their order.  Two contexts and a repeated
    call must give bit-identical energy, gradient, pattern, values and H.p (config 4 at 300 k pairs: ordinary rounds, split
    and long triangles, general rows through shared vertices are all present in the soup with a small vertex pool)."""
    from paper_2606_06511_b200 import inputs, tt
    dev = _dev()
    tdt = torch.float64 if dtype == "f64" else torch.float32
    pb = inputs.config4_sweep(n_tris=20_000, n_pairs=300_000)
    pos = torch.from_numpy(pb.pos).to(dev).to(tdt).contiguous()
    tris = torch.from_numpy(pb.tris).to(dev)
    prs = torch.from_numpy(pb.pairs).to(dev)
    p = torch.from_numpy(np.random.default_rng(3).normal(size=pb.pos.shape)).to(dev).to(tdt).contiguous()
    outs = []
    for rep in range(3):
        ctx = tt.Context(tdt, 1, 1.0, 0) if rep != 1 else ctx          # rep 1 reuses the first context
        out = tt.assemble(ctx, pos, tris, prs, want_hess=True)
        y = torch.empty_like(p)
        ctx.tt_hess_vec(out["prob"], p, y)
        torch.cuda.synchronize()
        outs.append((out["energy"].clone(), out["grad"].clone(), out["rowptr"].clone(), out["colind"].clone(), out["vals"].clone(), y))
    st = ctx.tt_stats()
    assert st["split_triangles"] + st["long_rounds"] > 0
    for o in outs[1:]:
        for a, b in zip(outs[0], o):
            assert a.shape == b.shape and torch.equal(a, b)
