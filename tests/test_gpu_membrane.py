"""GPU parity of the membrane term (tt_membrane_build / _energy_grad / _hess_vec and tt_newton_step / tt_untangle with
membrane = 1; SURVEY 8(f) NEXT-4 "with a simple membrane energy"; reading A18) against
oracle/membrane.py on the same seeded inputs, through the C ABI.  fp64: energy to 1e-13, gradient / H.p to 1e-12 of their
largest entry (both sides sum a vertex's few edges in fp64, in different orders); fp32: the same after rounding the inputs
to fp32 first -- the arithmetic is fp64 in both dtypes, so only the rounding of the OUTPUT vector is left (1e-6).  The
Newton step: discrete outcome equal, energies 1e-10, displacement 1e-7 (tests/test_gpu_newton.py's bar)."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

DEV = "cuda:0"


def crumpled(seed=11, subdiv=2):
    """Two icospheres (config 1's mesh, small); positions = rest scaled per vertex so edges are stretched AND compressed."""
    from paper_2606_06511_b200 import inputs
    pb = inputs.config1_icospheres(subdiv=subdiv)
    rng = np.random.default_rng(seed)
    rest = pb.pos.copy()
    pos = rest * (1.0 + 0.3 * rng.uniform(-1, 1, size=(rest.shape[0], 1))) + rng.normal(scale=0.02, size=rest.shape)
    return pb, rest, pos, rng


def ctx_for(dtype, mode=2):
    from paper_2606_06511_b200 import tt
    return tt.Context(dtype, mode, 1.0, 0)


@pytest.mark.parametrize("dtype", [torch.float64, torch.float32])
def test_energy_grad_hessvec_match_oracle(oracle_mod, dtype):
    from oracle import membrane as mb
    pb, rest, pos, rng = crumpled()
    # the mesh's triangles + duplicates of some (shared edges must still count once) + degenerate ones (i, i, j)
    tris = np.concatenate([pb.tris, pb.tris[:17], np.stack([pb.tris[:9, 0], pb.tris[:9, 0], pb.tris[:9, 2]], axis=1)]).astype(np.int32)
    p = rng.normal(size=pos.shape)
    if dtype == torch.float32:
        rest, pos, p = (a.astype(np.float32).astype(np.float64) for a in (rest, pos, p))
    k = 2.5
    Ed = mb.edges_of(tris)
    ln = np.linalg.norm(pos[Ed[:, 0]] - pos[Ed[:, 1]], axis=1)
    L = np.linalg.norm(rest[Ed[:, 0]] - rest[Ed[:, 1]], axis=1)
    assert (ln > L).any() and (ln < L).any()                       # the clamp is exercised both ways
    E_ref, g_ref = mb.energy_grad(pos, rest, tris, k)
    y_ref = mb.hess_vec(pos, rest, tris, k, p)
    ctx = ctx_for(dtype)
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(DEV).to(dtype).contiguous()
    ctx.tt_membrane_build(t(rest), torch.from_numpy(tris).to(DEV), k)
    e, g = ctx.tt_membrane_energy_grad(t(pos))
    y = ctx.tt_membrane_hess_vec(t(pos), t(p))
    e2, g2 = ctx.tt_membrane_energy_grad(t(pos), want_grad=False)
    torch.cuda.synchronize()
    tol = 1e-12 if dtype == torch.float64 else 1e-6
    assert abs(e.item() - E_ref) <= 1e-13 * E_ref and g2 is None and e2.item() == e.item()
    assert np.abs(g.cpu().double().numpy() - g_ref).max() <= tol * np.abs(g_ref).max()
    assert np.abs(y.cpu().double().numpy() - y_ref).max() <= tol * np.abs(y_ref).max()
    # rebuilt for another stiffness and another rest state: the context holds one membrane at a time
    ctx.tt_membrane_build(t(pos), torch.from_numpy(tris).to(DEV), 7.0)
    e0, g0 = ctx.tt_membrane_energy_grad(t(pos))
    assert e0.item() == 0.0 and not g0.any().item()                # at rest: nothing
    ctx.close()


def test_membrane_edge_cases():
    """No triangles, no vertices, coincident vertices (|d| = 0: the edge contributes nothing, results stay finite), calls
    without a build, the Newton step asking for a membrane of another mesh."""
    from paper_2606_06511_b200 import tt
    ctx = ctx_for(torch.float64)
    pos = torch.rand(5, 3, dtype=torch.float64, device=DEV)
    with pytest.raises(tt.TTError):
        ctx.tt_membrane_energy_grad(pos)
    with pytest.raises(tt.TTError):
        ctx.tt_membrane_hess_vec(pos, pos.clone())
    ctx.tt_membrane_build(pos, torch.zeros(0, 3, dtype=torch.int32, device=DEV), 1.0)
    e, g = ctx.tt_membrane_energy_grad(pos)
    assert e.item() == 0.0 and not g.any().item()
    assert not ctx.tt_membrane_hess_vec(pos, torch.ones_like(pos)).any().item()
    ctx.tt_membrane_build(pos[:0].contiguous(), torch.zeros(0, 3, dtype=torch.int32, device=DEV), 1.0)
    e, g = ctx.tt_membrane_energy_grad(pos[:0].contiguous())
    assert e.item() == 0.0 and g.shape == (0, 3)
    tris = torch.tensor([[0, 1, 2], [2, 1, 3]], dtype=torch.int32, device=DEV)
    rest = torch.tensor([[0, 0, 0], [1, 0, 0], [0, 1, 0], [1, 1, 0.0]], dtype=torch.float64, device=DEV)
    ctx.tt_membrane_build(rest, tris, 3.0)
    x = rest.clone()
    x[1] = x[0]                                                    # edge (0, 1) collapsed
    e, g = ctx.tt_membrane_energy_grad(x)
    y = ctx.tt_membrane_hess_vec(x, torch.ones_like(x) * torch.arange(4, device=DEV, dtype=torch.float64)[:, None])
    assert torch.isfinite(e).all() and torch.isfinite(g).all() and torch.isfinite(y).all()
    # vertex 0 feels only edge (0, 2): rest length 1, now still 1 -> no force on it from there
    assert g[0].abs().max().item() == 0.0
    with pytest.raises(tt.TTError):                                # the built mesh has 4 vertices, this one 5
        ctx.tt_newton_step(pos, tris, torch.zeros(0, 2, dtype=torch.int32, device=DEV), membrane=True)
    ctx.close()


@pytest.mark.parametrize("matrix_free", [False, True])
@pytest.mark.parametrize("k", [1.0, 50.0])
def test_newton_step_with_membrane_matches_oracle(oracle_mod, matrix_free, k):
    """5 inner steps: measured on this input, GPU and oracle agree to 1e-14 .. 1e-12 through step 5 and to 1e-8 (k = 1) /
    3e-6 (k = 50) at step 10, where the first Ritz values of the 120-unknown system have converged and CG's recurrences
    lose orthogonality (both implementations are correct to their own residual)."""
    from oracle import membrane as mb
    from paper_2606_06511_b200 import inputs
    from helpers import filter_margins
    pb = inputs.config0_soup(n_tris=48, pool=40, seed=5)
    pairs = filter_margins(oracle_mod, pb, 2)
    rng = np.random.default_rng(21)
    rest = pb.pos * (1.0 + 0.1 * rng.uniform(-1, 1, size=(pb.pos.shape[0], 1)))       # E_m, g_m != 0 at x
    ref = mb.newton_step(pb.pos, rest, pb.tris, pairs, k, hess_mode=2, mu=1e-2, pcg_iter=5, c1=1e-4, max_backtrack=20)
    ctx = ctx_for(torch.float64)
    pos = torch.from_numpy(pb.pos).to(DEV)
    tris = torch.from_numpy(pb.tris).to(DEV)
    ctx.tt_membrane_build(torch.from_numpy(rest).to(DEV), tris, k)
    rep = ctx.tt_newton_step(pos, tris, torch.from_numpy(pairs).to(DEV), mu=1e-2, pcg_iter=5, c1=1e-4, max_backtrack=20,
                             matrix_free=matrix_free, membrane=True)
    torch.cuda.synchronize()
    x = pos.cpu().numpy()
    ctx.close()
    assert rep["accepted"] == 1 and ref["accepted"] and rep["n_active"] == ref["n_active"] and rep["pcg_iters"] == 5
    assert rep["alpha"] == ref["alpha"] and rep["backtracks"] == ref["backtracks"]
    assert abs(rep["energy0"] - ref["E0"]) <= 1e-10 * ref["E0"]
    assert abs(rep["energy1"] - ref["E1"]) <= 1e-8 * ref["E0"]
    assert abs(rep["grad_norm"] - ref["gnorm"]) <= 1e-10 * ref["gnorm"]
    assert abs(rep["gd"] - ref["gd"]) <= 1e-8 * abs(ref["gd"])
    assert abs(rep["energy_membrane"] - mb.energy_grad(ref["x"], rest, pb.tris, k)[0]) <= 1e-8 * ref["E0"]
    dx, dx_ref = x - pb.pos, ref["x"] - pb.pos
    assert np.linalg.norm(dx - dx_ref) <= 1e-7 * np.linalg.norm(dx_ref)


def test_untangle_with_membrane(oracle_mod):
    """The demo on two interpenetrating icospheres: every step of the oracle's trajectory is reproduced from its own
    starting point (per-step parity: a long trajectory amplifies rounding, tests/test_gpu_newton.py); the GPU's own loop
    decreases E_T + E_m monotonically and keeps the edge strain far below the loop without the membrane."""
    from oracle import membrane as mb
    from paper_2606_06511_b200 import inputs
    pb = inputs.config1_icospheres(subdiv=2)
    k, kw = 1.0, dict(mu=1e-2, pcg_iter=8)
    ref = mb.untangle(pb.pos, pb.pos, pb.tris, k, inflate=0.05, max_steps=6, **kw)
    ctx = ctx_for(torch.float64)
    tris = torch.from_numpy(pb.tris).to(DEV)
    ctx.tt_membrane_build(torch.from_numpy(pb.pos).to(DEV), tris, k)
    for h in ref["history"]:
        pos = torch.from_numpy(np.ascontiguousarray(h["x0"])).to(DEV)
        rep = ctx.tt_untangle(pos, tris, inflate=0.05, max_steps=1, membrane=True, **kw)[0]
        assert rep["n_pairs"] == h["n_pairs"] and rep["n_active"] == h["n_active"] and rep["alpha"] == h["alpha"]
        assert abs(rep["energy0"] - h["E0"]) <= 1e-10 * h["E0"] and abs(rep["energy1"] - h["E1"]) <= 1e-8 * h["E0"]
        dx, dx_ref = pos.cpu().numpy() - h["x0"], h["x1"] - h["x0"]
        assert np.linalg.norm(dx - dx_ref) <= 1e-6 * np.linalg.norm(dx_ref)
    E = mb.edges_of(pb.tris)
    L = np.linalg.norm(pb.pos[E[:, 0]] - pb.pos[E[:, 1]], axis=1)
    strain = lambda x: np.abs(np.linalg.norm(x[E[:, 0]] - x[E[:, 1]], axis=1) / L - 1).max()
    pos = torch.from_numpy(pb.pos).to(DEV)
    ctx.tt_membrane_build(pos.clone(), tris, 100.0)
    hist = ctx.tt_untangle(pos, tris, inflate=0.05, max_steps=15, membrane=True, **kw)
    assert len(hist) == 15 and all(h["accepted"] for h in hist)
    assert all(h["energy1"] < h["energy0"] for h in hist)
    free = torch.from_numpy(pb.pos).to(DEV)
    hist0 = ctx.tt_untangle(free, tris, inflate=0.05, max_steps=15, **kw)
    assert len(hist0) >= 1
    assert strain(pos.cpu().numpy()) < 0.2 * strain(free.cpu().numpy())
    ctx.close()
