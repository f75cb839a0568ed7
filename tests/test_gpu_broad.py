"""Broad phase through the C ABI against the oracle's all-pairs definition.
Integer output: bit-exact (the candidate set is unique and the order is canonical, lexicographic)."""
import numpy as np
import pytest
import torch

pytestmark = pytest.mark.gpu


def gpu_pairs(pos_np, tris_np, inflate, dtype="f64"):
    from paper_2606_06511_b200 import tt
    dev = torch.device("cuda:0")
    tdt = torch.float64 if dtype == "f64" else torch.float32
    ctx = tt.Context(tdt, 1, 1.0, 0)
    pos = torch.from_numpy(np.ascontiguousarray(pos_np)).to(dev).to(tdt).contiguous()
    tris = torch.from_numpy(np.ascontiguousarray(tris_np)).to(dev)
    out = ctx.tt_broad_phase(pos, tris, inflate)
    torch.cuda.synchronize()
    res = out.cpu().numpy()
    ctx.close()
    return res


def check(oracle, pos, tris, inflate, dtype="f64"):
    pos_o = pos.astype(np.float32).astype(np.float64) if dtype == "f32" else pos   # the oracle sees the stored values
    ref = oracle.broad_phase(pos_o, tris, inflate)
    got = gpu_pairs(pos, tris, inflate, dtype)
    assert got.shape == ref.shape, (got.shape, ref.shape)
    assert (got == ref).all()
    return ref


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_icospheres_and_cloth(oracle_mod, dtype):
    from paper_2606_06511_b200 import inputs
    ico = inputs.config1_icospheres()
    assert check(oracle_mod, ico.pos, ico.tris, 0.02, dtype).shape[0] > 40_000
    assert check(oracle_mod, ico.pos, ico.tris, 0.0, dtype).shape[0] > 1_000
    cloth = inputs.config2_cloth(n=96)                       # 18k triangles, several CTAs, ragged tail
    assert check(oracle_mod, cloth.pos, cloth.tris, 0.002, dtype).shape[0] > 10_000


def test_soup_with_size_spread(oracle_mod):
    """Random soup whose triangle sizes differ by 30x: the cell (= largest box) holds many small boxes."""
    rng = np.random.default_rng(3)
    n = 3000
    c = rng.uniform(0, 1, (n, 1, 3))
    size = np.where(rng.uniform(size=(n, 1, 1)) < 0.02, 0.3, 0.01)
    pos = (c + size * rng.normal(size=(n, 3, 3))).reshape(-1, 3)
    tris = np.arange(3 * n, dtype=np.int32).reshape(n, 3)
    assert check(oracle_mod, pos, tris, 0.0).shape[0] > 1000
    # shared-vertex pairs are dropped: draw the ids from a small pool
    pool = rng.integers(0, 400, size=(n, 3)).astype(np.int32)
    pool = pool[(pool[:, 0] != pool[:, 1]) & (pool[:, 1] != pool[:, 2]) & (pool[:, 0] != pool[:, 2])]
    check(oracle_mod, rng.uniform(0, 1, (400, 3)), pool[:600], 0.0)


def test_edge_cases(oracle_mod):
    tri = np.array([[0, 0, 0], [1, 0, 0], [0, 1, 0]], dtype=np.float64)
    one = np.array([[0, 1, 2]], dtype=np.int32)
    assert gpu_pairs(tri, one, 0.0).shape == (0, 2)                       # a single triangle
    assert gpu_pairs(tri, np.zeros((0, 3), dtype=np.int32), 0.0).shape == (0, 2)
    pos = np.concatenate([tri, tri + np.array([1.0, 0, 0]), tri + np.array([1.5, 0, 0]) + np.array([1.0, 0, 0])])
    tris = np.arange(9, dtype=np.int32).reshape(3, 3)
    assert check(oracle_mod, pos, tris, 0.0).tolist() == [[0, 1]]         # touching boxes count (closed)
    assert check(oracle_mod, pos, tris, 0.25).tolist() == [[0, 1], [1, 2]]  # the 0.5 gap closes at 2 * 0.25
    flat = np.zeros((6, 3))                                               # all boxes degenerate to a point
    assert check(oracle_mod, flat, np.arange(6, dtype=np.int32).reshape(2, 3), 0.0).tolist() == [[0, 1]]


def test_full_size_sampled(oracle_mod):
    """Config 2 at full size (130 050 triangles, ~1 M candidates): the whole list against the
    generators' grid routine is NOT the check (that is not the oracle); instead the partners of
    sampled triangles are recomputed by the oracle's definition (all nT boxes tested against the
    sample) and must equal the GPU's, and the list must be strictly lexicographic."""
    from paper_2606_06511_b200 import inputs
    rng = np.random.default_rng(5)
    pb = inputs.config2_cloth()
    inflate = 0.002
    got = gpu_pairs(pb.pos, pb.tris, inflate)
    nT = pb.tris.shape[0]
    key = got[:, 0].astype(np.int64) * nT + got[:, 1]
    assert (got[:, 0] < got[:, 1]).all() and (np.diff(key) > 0).all()
    assert abs(got.shape[0] - 1_000_000) < 100_000
    P = pb.pos[pb.tris]
    lo, hi = P.min(axis=1) - inflate, P.max(axis=1) + inflate
    for t in rng.choice(nT, size=200, replace=False):
        ov = ((lo[t] <= hi) & (lo <= hi[t])).all(axis=1)
        adj = (pb.tris[:, :, None] == pb.tris[t][None, None, :]).any(axis=(1, 2))
        partners = np.nonzero(ov & ~adj)[0]
        partners = partners[partners != t]
        mine = np.concatenate([got[got[:, 0] == t, 1], got[got[:, 1] == t, 0]])
        assert np.array_equal(np.sort(mine), partners)


def test_pairs_feed_the_hot_path(oracle_mod):
    """The device list goes into tt_problem: energy of the broad phase's candidates == oracle.  The
    broad phase (unlike the generators) applies no margins, so the pairs within the G-margins of a
    discrete decision are dropped from BOTH sides first: the exact active count
    is only demanded of pairs the bit-exactness contract covers."""
    from helpers import filter_margins
    from paper_2606_06511_b200 import inputs, tt
    dev = torch.device("cuda:0")
    pb = inputs.config1_icospheres()
    ctx = tt.Context(torch.float64, 1, 1.0, 0)
    pos = torch.from_numpy(pb.pos).to(dev)
    tris = torch.from_numpy(pb.tris).to(dev)
    pairs = ctx.tt_broad_phase(pos, tris, 0.02)
    cand = oracle_mod.broad_phase(pb.pos, pb.tris, 0.02)
    assert (pairs.cpu().numpy() == cand).all()
    _, degenerate = inputs.classify_pairs(pb.pos, pb.tris, cand, 1e-6)
    kept = filter_margins(oracle_mod, inputs.Problem(pb.pos, pb.tris, np.ascontiguousarray(cand[~degenerate])), 1)
    key = cand[:, 0].astype(np.int64) * pb.n_tris + cand[:, 1]
    keep = np.isin(key, kept[:, 0].astype(np.int64) * pb.n_tris + kept[:, 1])
    assert keep.sum() == kept.shape[0] and keep.sum() > 0.9 * cand.shape[0]
    pairs = pairs[torch.from_numpy(keep).to(dev)].contiguous()      # still the broad phase's device array
    prob = ctx.problem(pos, tris, pairs)
    e = torch.zeros(1, dtype=torch.float64, device=dev)
    na = torch.zeros(1, dtype=torch.int64, device=dev)
    ctx.tt_energy(prob, e, None, None, None, na)
    torch.cuda.synchronize()
    ref = oracle_mod.pairs(pb.pos, pb.tris, kept, 1.0, want_J=False)
    assert int(na.cpu()[0]) == int(ref["active"].sum())
    assert abs(float(e.cpu()[0]) - ref["T"].sum()) <= 1e-9 * ref["T"].sum()
    ctx.close()
