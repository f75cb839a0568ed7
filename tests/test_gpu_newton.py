"""GPU parity of the consumer loop (tt_newton_step, tt_untangle; SURVEY 8(f) NEXT-2 line search, NEXT-4; PAPER.md L5, L41-43;
DESIGN.md reading A16) against oracle/newton.py on the same seeded inputs, through the C ABI.  The discrete outcome (accepted
step length = number of halvings, inner iteration count, active count) must be equal; energies agree to 1e-10 / gradient-
derived scalars to 1e-9; the DISPLACEMENT x_new - x (not the position, which would hide it) to 1e-7 -- the direction is a
20-step PCG iterate, which amplifies the 1e-10 differences of its inputs."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu


def gpu_step(pb_pos, tris_np, pairs_np, dtype=torch.float64, mode=2, **kw):
    from paper_2606_06511_b200 import tt
    dev = torch.device("cuda:0")
    ctx = tt.Context(dtype, mode, 1.0, 0)
    pos = torch.from_numpy(pb_pos).to(dev).to(dtype).contiguous()
    tris = torch.from_numpy(tris_np).to(dev)
    prs = torch.from_numpy(pairs_np).to(dev)
    rep = ctx.tt_newton_step(pos, tris, prs, **kw)
    torch.cuda.synchronize()
    x = pos.cpu().numpy().astype(np.float64)
    ctx.close()
    return rep, x


@pytest.mark.parametrize("mode,mu", [(2, 1e-3), (2, 1e-1), (3, 1e-2)])
def test_newton_step_matches_oracle(oracle_mod, mode, mu):
    from oracle import newton
    from paper_2606_06511_b200 import inputs
    from helpers import filter_margins
    pb = inputs.config0_soup()
    pairs = filter_margins(oracle_mod, pb, mode)
    ref = newton.newton_step(pb.pos, pb.tris, pairs, hess_mode=mode, mu=mu, pcg_iter=20, c1=1e-4, max_backtrack=20)
    rep, x = gpu_step(pb.pos, pb.tris, pairs, mode=mode, mu=mu, pcg_iter=20, c1=1e-4, max_backtrack=20)
    assert rep["accepted"] == 1 and ref["accepted"]
    assert rep["n_active"] == ref["n_active"] and rep["pcg_iters"] == ref["pcg_iters"] == 20
    assert rep["alpha"] == ref["alpha"] and rep["backtracks"] == ref["backtracks"]
    assert abs(rep["energy0"] - ref["E0"]) <= 1e-10 * ref["E0"]
    assert abs(rep["energy1"] - ref["E1"]) <= 1e-8 * ref["E0"]
    assert abs(rep["grad_norm"] - ref["gnorm"]) <= 1e-10 * ref["gnorm"]
    assert abs(rep["gd"] - ref["gd"]) <= 1e-8 * abs(ref["gd"])
    dx, dx_ref = x - pb.pos, ref["x"] - pb.pos
    assert np.linalg.norm(dx - dx_ref) <= 1e-7 * np.linalg.norm(dx_ref)
    assert rep["energy1"] < rep["energy0"]


def test_newton_step_matrix_free_and_fp32(oracle_mod):
    """matrix_free = 1: plain CG on tt_hess_vec (no preconditioner) -- compared with the oracle's un-preconditioned CG
    direction; fp32: same discrete outcome, displacement to 1e-3."""
    from oracle import newton
    from paper_2606_06511_b200 import inputs
    from helpers import filter_margins
    pb = inputs.config0_soup()
    pairs = filter_margins(oracle_mod, pb, 2)
    r = oracle_mod.assemble(pb.pos, pb.tris, pairs, 1.0, 2)
    # plain CG amplifies summation-order differences quickly on a badly scaled system (tests/test_gpu_solve.py): shift =
    # the mean diagonal, 5 steps
    rowv = np.repeat(np.arange(pb.n_verts), np.diff(r["rowptr"]))
    mu = float(np.mean([np.trace(b) for b in r["vals"][r["colind"] == rowv]])) / 3
    sol = oracle_mod.pcg(r["rowptr"], r["colind"], r["vals"], r["grad"], shift=mu, max_iter=5, rtol=0.0, precond=False)
    rep, x = gpu_step(pb.pos, pb.tris, pairs, mode=2, mu=mu, pcg_iter=5, matrix_free=True)
    assert rep["accepted"] == 1 and rep["nnzb"] == r["nnzb"]
    d_gpu = (pb.pos - x) / rep["alpha"]
    assert np.linalg.norm(d_gpu - sol["x"]) <= 1e-7 * np.linalg.norm(sol["x"])
    pos32 = pb.pos.astype(np.float32).astype(np.float64)
    pb32 = type(pb)(pos32, pb.tris, pb.pairs, pb.name, pb.meta)
    pairs32 = filter_margins(oracle_mod, pb32, 2)
    ref = newton.newton_step(pos32, pb.tris, pairs32, hess_mode=2, mu=1e-2, pcg_iter=10)
    rep, x = gpu_step(pos32, pb.tris, pairs32, dtype=torch.float32, mode=2, mu=1e-2, pcg_iter=10)
    assert rep["accepted"] == 1 and rep["alpha"] == ref["alpha"] and rep["n_active"] == ref["n_active"]
    assert abs(rep["energy1"] - ref["E1"]) <= 1e-4 * ref["E0"]
    assert np.linalg.norm((x - pos32) - (ref["x"] - pos32)) <= 2e-3 * np.linalg.norm(ref["x"] - pos32)


def test_newton_step_edge_cases(oracle_mod):
    from paper_2606_06511_b200 import inputs, tt
    pb = inputs.config0_soup()
    # nothing active: accepted, positions untouched, energy 0
    far = np.array([[0, 1]], dtype=np.int32)
    pos = pb.pos.copy()
    pos[3:6] += 100.0
    rep, x = gpu_step(pos, pb.tris, far)
    assert rep["accepted"] == 1 and rep["n_active"] == 0 and rep["alpha"] == 0.0 and (x == pos).all()
    # impossible Armijo constant with no halvings allowed: rejected, positions untouched
    rep, x = gpu_step(pb.pos, pb.tris, pb.pairs, mu=1e-9, pcg_iter=3, c1=0.999999, max_backtrack=0)
    assert rep["accepted"] == 0 and (x == pb.pos).all() and rep["backtracks"] == 1 and rep["energy1"] == rep["energy0"]
    # bad options
    dev = torch.device("cuda:0")
    ctx = tt.Context(torch.float64, 2, 1.0, 0)
    p = torch.from_numpy(pb.pos).to(dev)
    with pytest.raises(tt.TTError):
        ctx.tt_newton_step(p, torch.from_numpy(pb.tris).to(dev), torch.from_numpy(pb.pairs).to(dev), mu=0.0)
    ctx.close()


def sheets(n=4, seed=5):
    rng = np.random.default_rng(seed)
    u, v = np.meshgrid(np.linspace(0, 1, n), np.linspace(0, 1, n), indexing="ij")
    quad = lambda i, j: i * n + j
    tr = []
    for i in range(n - 1):
        for j in range(n - 1):
            tr += [[quad(i, j), quad(i + 1, j), quad(i + 1, j + 1)], [quad(i, j), quad(i + 1, j + 1), quad(i, j + 1)]]
    tr = np.array(tr, dtype=np.int32)
    a = np.stack([u.ravel(), v.ravel(), 0.06 * np.sin(3 * u.ravel())], axis=1)
    b = np.stack([u.ravel() + 0.013, v.ravel() + 0.021, 0.02 - 0.05 * np.sin(3 * u.ravel() + 0.4)], axis=1)
    pos = np.concatenate([a, b]) + rng.normal(scale=1e-3, size=(2 * n * n, 3))
    return pos, np.concatenate([tr, tr + n * n]).astype(np.int32)


def test_untangle_matches_oracle_trajectory(oracle_mod):
    """The whole loop (GPU broad phase + step) on the two crossing sheets of tests/test_oracle_newton.py, 8 steps with a
    6-step inner solve and mu = 0.1.
    (1) Step by step along the ORACLE's trajectory: from each of its iterates x_k one GPU loop step must reproduce the
        oracle's step k -- candidate count, active count and step length equal, E0 to 1e-10, E1 to 1e-9, displacement to
        1e-8.  Nothing compounds, so the late steps are held to the same bar as the first.
    (2) Free running: same discrete outcomes at every step, energies to 1e-6, final positions to 1e-6 of the path length.
    Why few inner steps: |H| / mu is 1e5-1e6 here and two correct CG implementations drift apart as CG loses
    orthogonality -- measured on this system, oracle vs GPU: 1e-12 after 10 steps, 5e-10 after 20, 2e-5 after 30."""
    from oracle import newton
    from paper_2606_06511_b200 import tt
    pos_np, tris_np = sheets()
    kw = dict(inflate=0.05, mu=0.1, pcg_iter=6)
    ref = newton.untangle(pos_np, tris_np, max_steps=8, hess_mode=2, **kw)
    h_ref = ref["history"]
    assert len(h_ref) == 8 and all(b["accepted"] for b in h_ref)
    dev = torch.device("cuda:0")
    ctx = tt.Context(torch.float64, 2, 1.0, 0)
    tris = torch.from_numpy(tris_np).to(dev)
    for k, b in enumerate(h_ref):
        pos = torch.from_numpy(b["x0"]).to(dev).contiguous()
        (a,) = ctx.tt_untangle(pos, tris, max_steps=1, **kw)
        assert a["n_pairs"] == b["n_pairs"] and a["n_active"] == b["n_active"] and a["alpha"] == b["alpha"], k
        assert abs(a["energy0"] - b["E0"]) <= 1e-10 * b["E0"], k
        assert abs(a["energy1"] - b["E1"]) <= 1e-9 * b["E0"], k
        dx, dx_ref = pos.cpu().numpy() - b["x0"], b["x1"] - b["x0"]
        assert np.linalg.norm(dx - dx_ref) <= 1e-8 * np.linalg.norm(dx_ref), k
    pos = torch.from_numpy(pos_np).to(dev)
    hist = ctx.tt_untangle(pos, tris, max_steps=8, **kw)
    torch.cuda.synchronize()
    assert len(hist) == 8
    path = sum(np.linalg.norm(b["x1"] - b["x0"]) for b in h_ref)
    for a, b in zip(hist, h_ref):
        assert a["n_pairs"] == b["n_pairs"] and a["n_active"] == b["n_active"] and a["alpha"] == b["alpha"]
        assert abs(a["energy0"] - b["E0"]) <= 1e-6 * b["E0"] and a["energy1"] < a["energy0"]
    assert np.linalg.norm(pos.cpu().numpy() - h_ref[-1]["x1"]) <= 1e-6 * path
    assert hist[-1]["energy1"] < 0.5 * hist[0]["energy0"]
    ctx.close()


def test_untangle_ends_intersection_free(oracle_mod):
    """The loop with the parameters of tests/test_oracle_newton.py's untangling run (mu = 1e-2, 30 inner steps): it stops
    because no pair is active, and the ORACLE's broad phase + Moeller test on the GPU's final positions agrees."""
    from paper_2606_06511_b200 import tt
    pos_np, tris_np = sheets()
    dev = torch.device("cuda:0")
    ctx = tt.Context(torch.float64, 2, 1.0, 0)
    pos = torch.from_numpy(pos_np).to(dev)
    hist = ctx.tt_untangle(pos, torch.from_numpy(tris_np).to(dev), inflate=0.05, max_steps=60, mu=1e-2, pcg_iter=30)
    torch.cuda.synchronize()
    assert hist[-1]["n_active"] == 0 and all(h["accepted"] for h in hist) and len(hist) < 60
    assert all(h["energy1"] <= h["energy0"] for h in hist)
    x = pos.cpu().numpy()
    cand = oracle_mod.broad_phase(x, tris_np, 0.05)
    assert oracle_mod.pairs(x, tris_np, cand, 1.0, want_J=False)["active"].sum() == 0
    ctx.close()


def test_untangle_icospheres_energy_falls():
    """configs[1] (two interpenetrating icospheres): 8 steps of the loop, energy strictly decreasing, every step accepted."""
    from paper_2606_06511_b200 import inputs, tt
    pb = inputs.config1_icospheres()
    dev = torch.device("cuda:0")
    ctx = tt.Context(torch.float64, 2, 1.0, 0)
    pos = torch.from_numpy(pb.pos).to(dev)
    hist = ctx.tt_untangle(pos, torch.from_numpy(pb.tris).to(dev), inflate=0.02, max_steps=8, mu=1e-4, pcg_iter=30)
    assert len(hist) >= 2 and all(h["accepted"] for h in hist)
    assert all(h["energy1"] < h["energy0"] for h in hist if h["n_active"] > 0)
    assert hist[-1]["energy1"] < 0.6 * hist[0]["energy0"]
    ctx.close()
