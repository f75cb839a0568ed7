"""GPU parity of the consumer of the assembly: tt_bsr_spmv, tt_block_jacobi and
tt_pcg_solve (assembled and matrix-free back ends) through the C ABI against the oracle's textbook
definitions (oracle.bsr_matvec, oracle.block_jacobi, oracle.pcg), on the same seeded inputs.

Tolerances: the product is a single evaluation -- 1e-12 per row in fp64; a 3x3 inverse agrees to
2e-12 x cond(block) (+ the fp32 rounding of the output in the fp32 variant).  CG iterates amplify rounding differences (different summation trees) with the step
count: x_k agrees to 1e-10 at k = 1, 1e-9 at k = 5 and 1e-6 at k = 20, relative to |x_k|, with the
block-Jacobi preconditioner; plain CG on these badly scaled systems is far more sensitive to the summation
order (measured 8e-5 on the 196 k-unknown cloth after 20 steps) and gets 1e-8 / 1e-2 (a sanity bound, not a parity claim).  The step count at a
given rtol is exact away from ties (+-1)."""
import numpy as np
import pytest

from helpers import filter_margins, rel

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu


def assembled(oracle, pb, dtype="f64", hess_mode=2):
    from paper_2606_06511_b200 import tt
    dev = torch.device("cuda:0")
    tdt = torch.float64 if dtype == "f64" else torch.float32
    pos_np = pb.pos.astype(np.float32).astype(np.float64) if dtype == "f32" else pb.pos
    pairs = filter_margins(oracle, type(pb)(pos_np, pb.tris, pb.pairs, pb.name, pb.meta), hess_mode)
    ref = oracle.assemble(pos_np, pb.tris, pairs, 1.0, hess_mode)
    ctx = tt.Context(tdt, hess_mode, 1.0, 0)
    pos = torch.from_numpy(pos_np).to(dev).to(tdt).contiguous()
    out = tt.assemble(ctx, pos, torch.from_numpy(pb.tris).to(dev), torch.from_numpy(pairs).to(dev))
    torch.cuda.synchronize()
    assert out["nnzb"] == ref["nnzb"]
    return ctx, ref, out, tdt, dev


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_bsr_spmv_and_block_jacobi(oracle_mod, dtype):
    from paper_2606_06511_b200 import inputs
    for pb in (inputs.config0_soup(), inputs.config1_icospheres(), inputs.config4_sweep(n_tris=30_000, n_pairs=150_000)):
        ctx, ref, out, tdt, dev = assembled(oracle_mod, pb, dtype)
        nV = pb.n_verts
        # the ORACLE's matrix on both sides (rounded to the storage type): the product alone is under test
        vals_np = ref["vals"].astype(np.float32).astype(np.float64) if dtype == "f32" else ref["vals"]
        x_np = np.random.default_rng(3).normal(size=(nV, 3))
        if dtype == "f32":
            x_np = x_np.astype(np.float32).astype(np.float64)
        rp = torch.from_numpy(ref["rowptr"]).to(dev)
        ci = torch.from_numpy(ref["colind"]).to(dev)
        va = torch.from_numpy(vals_np).to(dev).to(tdt)
        x = torch.from_numpy(x_np).to(dev).to(tdt)
        y = torch.full_like(x, float("nan"))
        for shift in (0.0, 0.37):
            ctx.tt_bsr_spmv(rp, ci, va, x, y, shift)
            torch.cuda.synchronize()
            y_ref = oracle_mod.bsr_matvec(ref["rowptr"], ref["colind"], vals_np, x_np) + shift * x_np
            assert rel(y.cpu().numpy(), y_ref) <= (1e-13 if dtype == "f64" else 1e-6)
            scale = np.zeros(nV)
            row_of = np.repeat(np.arange(nV), np.diff(ref["rowptr"]))
            np.add.at(scale, row_of, np.linalg.norm(vals_np.reshape(-1, 9), axis=1) * np.linalg.norm(x_np[ref["colind"]], axis=1))
            scale += shift * np.linalg.norm(x_np, axis=1)
            d = np.linalg.norm(y.cpu().numpy() - y_ref, axis=1)
            assert (d[scale > 0] / scale[scale > 0]).max() <= (1e-12 if dtype == "f64" else 1e-5)   # every row on its own scale
            assert not y.cpu().numpy()[scale == 0].any()
        mean_diag = float(np.mean([np.trace(b) for b in vals_np[ref["colind"] == row_of]])) / 3 if ref["nnzb"] else 1.0
        for shift in (1e-2 * mean_diag, mean_diag):
            minv = torch.full((nV, 3, 3), float("nan"), dtype=tdt, device=dev)
            ctx.tt_block_jacobi(rp, ci, va, minv, shift)
            torch.cuda.synchronize()
            m_ref = oracle_mod.block_jacobi(ref["rowptr"], ref["colind"], vals_np, shift)
            m = minv.cpu().numpy().astype(np.float64)
            err = np.linalg.norm((m - m_ref).reshape(nV, 9), axis=1) / np.linalg.norm(m_ref.reshape(nV, 9), axis=1)
            # every block on its own norm; an inverse is only defined to cond(block) x eps (the oracle's
            # Gauss-Jordan and the GPU's cofactors are both backward stable, not identical)
            cond = np.linalg.cond(m_ref)
            assert (err <= 2e-12 * cond + (1e-12 if dtype == "f64" else 2e-7)).all(), float((err / cond).max())
        ctx.close()


@pytest.mark.parametrize("backend", ["bsr", "matrix_free"])
@pytest.mark.parametrize("precond", [True, False])
def test_pcg_iterates_match_oracle(oracle_mod, backend, precond):
    """x_k after k = 1, 5, 20 steps of (H + mu I) x = -grad on configs 0-2 (PSD2), fp64."""
    from paper_2606_06511_b200 import inputs
    for pb in (inputs.config0_soup(), inputs.config1_icospheres(), inputs.config2_cloth()):
        ctx, ref, out, tdt, dev = assembled(oracle_mod, pb, "f64", 2)
        nV = pb.n_verts
        rowv = np.repeat(np.arange(nV), np.diff(ref["rowptr"]))
        # mu = 1 % of the mean diagonal with the preconditioner; the mean diagonal itself for plain CG (whose
        # iterates on the badly scaled 1 % system differ by 1e-4 between two summation orders after 20 steps:
        # a property of CG in floating point, not of either implementation)
        mu = (1e-2 if precond else 1.0) * float(np.mean([np.trace(b) for b in ref["vals"][ref["colind"] == rowv]])) / 3
        b_np = -ref["grad"]
        b = torch.from_numpy(b_np).to(dev)
        x = torch.full_like(b, float("nan"))
        minv = None
        if precond:
            minv = torch.empty((nV, 3, 3), dtype=tdt, device=dev)
            ctx.tt_block_jacobi(out["rowptr"], out["colind"], out["vals"], minv, mu)
        orc = oracle_mod.pcg(ref["rowptr"], ref["colind"], ref["vals"], b_np, mu, 20, 0.0, precond=precond, history=True)
        for k, tol in ((1, 1e-10), (5, 1e-9 if precond else 1e-8), (20, 1e-6 if precond else 1e-2)):
            kw = dict(rowptr=out["rowptr"], colind=out["colind"], vals=out["vals"]) if backend == "bsr" else {}
            iters, relres = ctx.tt_pcg_solve(out["prob"], b, x, minv=minv, max_iter=k, rtol=0.0, shift=mu, **kw)
            torch.cuda.synchronize()
            assert iters == k
            assert rel(x.cpu().numpy(), orc["x_hist"][k]) <= tol, (pb.name, k)
            assert abs(relres - orc["res"][k] / orc["res"][0]) <= max(1e-6, 20 * tol) * (orc["res"][k] / orc["res"][0]) + 1e-14
        ctx.close()


def test_pcg_converges_and_stops_like_the_oracle(oracle_mod):
    """rtol stop: same step count as the oracle, solution equal to numpy.linalg.solve on config 0's dense
    576 x 576 regularised system; the iterate does not depend on check_every; b = 0 returns x = 0 in 0 steps."""
    from paper_2606_06511_b200 import inputs
    pb = inputs.config0_soup()
    ctx, ref, out, tdt, dev = assembled(oracle_mod, pb, "f64", 2)
    nV = pb.n_verts
    H = np.zeros((3 * nV, 3 * nV))
    for r in range(nV):
        for e in range(ref["rowptr"][r], ref["rowptr"][r + 1]):
            H[3 * r:3 * r + 3, 3 * ref["colind"][e]:3 * ref["colind"][e] + 3] += ref["vals"][e]
    mu = 1e-2 * np.trace(H) / (3 * nV)
    b_np = -ref["grad"]
    x_star = np.linalg.solve(H + mu * np.eye(3 * nV), b_np.ravel()).reshape(nV, 3)
    b = torch.from_numpy(b_np).to(dev)
    minv = torch.empty((nV, 3, 3), dtype=tdt, device=dev)
    ctx.tt_block_jacobi(out["rowptr"], out["colind"], out["vals"], minv, mu)
    orc = oracle_mod.pcg(ref["rowptr"], ref["colind"], ref["vals"], b_np, mu, 2000, 1e-8, precond=True)
    xs = []
    for ce in (1, 7, 0):
        x = torch.full_like(b, float("nan"))
        iters, relres = ctx.tt_pcg_solve(out["prob"], b, x, out["rowptr"], out["colind"], out["vals"], minv, max_iter=2000,
                                         rtol=1e-8, shift=mu, check_every=ce)
        assert abs(iters - orc["iters"]) <= max(1, orc["iters"] // 50) and relres <= 1e-8   # ~290 steps: within 2 %
        assert rel(x.cpu().numpy(), x_star) <= 1e-6
        xs.append(x.cpu().numpy())
    assert (xs[0] == xs[1]).all() and (xs[0] == xs[2]).all()
    # matrix-free back end: same answer without ever forming a block
    x = torch.full_like(b, float("nan"))
    iters, relres = ctx.tt_pcg_solve(out["prob"], b, x, minv=minv, max_iter=2000, rtol=1e-8, shift=mu)
    assert abs(iters - orc["iters"]) <= max(1, orc["iters"] // 50) and rel(x.cpu().numpy(), x_star) <= 1e-6
    # b = 0
    iters, relres = ctx.tt_pcg_solve(out["prob"], torch.zeros_like(b), x, out["rowptr"], out["colind"], out["vals"], minv,
                                     max_iter=10, rtol=1e-8, shift=mu)
    assert iters == 0 and not x.cpu().numpy().any()
    ctx.close()


def test_pcg_fp32_variant(oracle_mod):
    """fp32 storage of matrix and vectors (scalars and dot products stay fp64): 1e-3 on the early iterates."""
    from paper_2606_06511_b200 import inputs
    pb = inputs.config4_sweep(n_tris=30_000, n_pairs=150_000)
    ctx, ref, out, tdt, dev = assembled(oracle_mod, pb, "f32", 2)
    nV = pb.n_verts
    rowv = np.repeat(np.arange(nV), np.diff(ref["rowptr"]))
    mu = 0.1 * float(np.mean([np.trace(b) for b in ref["vals"][ref["colind"] == rowv]])) / 3
    b_np = (-ref["grad"]).astype(np.float32).astype(np.float64)
    b = torch.from_numpy(b_np).to(dev).to(tdt)
    x = torch.empty_like(b)
    minv = torch.empty((nV, 3, 3), dtype=tdt, device=dev)
    ctx.tt_block_jacobi(out["rowptr"], out["colind"], out["vals"], minv, mu)
    orc = oracle_mod.pcg(ref["rowptr"], ref["colind"], ref["vals"], b_np, mu, 5, 0.0, precond=True, history=True)
    for k in (1, 5):
        ctx.tt_pcg_solve(out["prob"], b, x, out["rowptr"], out["colind"], out["vals"], minv, max_iter=k, shift=mu)
        assert rel(x.cpu().numpy(), orc["x_hist"][k]) <= 1e-3
    ctx.close()
