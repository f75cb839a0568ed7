"""tt_energy_static (include/tt.h): the allocation-free variant of tt_energy -- K1's per-CTA partials and counts in a
file-scope device array of the library instead of the context's workspace.  Collected LAST on purpose (the name sorts
after every other test file): the suite runs with pytest -x, and a failure here must not hide the parity tests.

Checked against the EXISTING path (tt_energy) on the same inputs: same active count, energy within the tolerance the
parity tests use for the total energy (tests/test_gpu_parity.py TOL["e"]: 1e-10 fp64, the fp32 figure below; the two are
in fact bit-identical, which is asserted too),
on two calls in a row that share the array -- a large problem first, a smaller one second, so stale partials of the first
would show up in the second -- and once more for the large one.  Also: the size limit is an error, not a launch; nothing
is allocated by the call (torch's view of the device's free memory does not move); both dtypes."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

DEV = "cuda:0"
TOL_E = {"f64": 1e-10, "f32": 1e-4}   # tests/test_gpu_parity.py TOL[dtype]["e"]
TT_ERR_CAPACITY = -4                  # include/tt.h


def _problem(ctx, pb, tdt):
    pos = torch.from_numpy(pb.pos).to(DEV).to(tdt).contiguous()
    tris = torch.from_numpy(pb.tris).to(DEV)
    prs = torch.from_numpy(pb.pairs).to(DEV)
    return ctx.problem(pos, tris, prs)


def _existing(ctx, prob, tdt):
    e = torch.zeros(1, dtype=tdt, device=DEV)
    na = torch.zeros(1, dtype=torch.int64, device=DEV)
    ctx.tt_energy(prob, e, None, None, None, na)
    torch.cuda.synchronize()
    return e.cpu().double().item(), int(na.item())


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_energy_static_matches_tt_energy_on_calls_in_a_row(dtype):
    from paper_2606_06511_b200 import inputs, tt
    tdt = torch.float64 if dtype == "f64" else torch.float32
    small = inputs.config4_sweep(n_tris=20_000, n_pairs=300_000)       # 2 344 CTAs of K1: one-level final sum
    # the same mesh with its candidate list repeated 30 x (duplicates are legal input and add): 70 313 CTAs, two levels
    big = type(small)(small.pos, small.tris, np.ascontiguousarray(np.tile(small.pairs, (30, 1))), "config4 x30", small.meta)
    tiny = inputs.config0_soup()
    ctx = tt.Context(tdt, 1, 1.0, 0)
    probs = [_problem(ctx, pb, tdt) for pb in (big, small, tiny)]
    refs = [_existing(ctx, p, tdt) for p in probs]
    assert refs[0][1] > 1_000_000 and refs[1][1] > 10_000 and refs[2][1] > 0
    ctx2 = tt.Context(tdt, 1, 1.0, 0)                                  # a fresh context: its workspace is never grown
    e = torch.full((1,), -1.0, dtype=tdt, device=DEV)
    na = torch.full((1,), -1, dtype=torch.int64, device=DEV)
    outs = [(torch.zeros(1, dtype=tdt, device=DEV), torch.zeros(1, dtype=torch.int64, device=DEV)) for _ in range(2)]
    ctx2.tt_energy_static(probs[2], e, na)      # first launch of the new kernels: the driver loads their code lazily
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    # calls in a row on one stream, sharing the static array: big, small, tiny, big again
    for i in (0, 1, 2, 0, 1):
        ctx2.tt_energy_static(probs[i], e, na)
        torch.cuda.synchronize()
        got_e, got_n = e.cpu().double().item(), int(na.item())
        assert got_n == refs[i][1]
        assert abs(got_e - refs[i][0]) <= TOL_E[dtype] * abs(refs[i][0])
        assert got_e == refs[i][0]                                     # same partials, same summation order
    # back to back WITHOUT a synchronisation in between (same stream: ordered), outputs in separate buffers
    ctx2.tt_energy_static(probs[0], outs[0][0], outs[0][1])
    ctx2.tt_energy_static(probs[1], outs[1][0], outs[1][1])
    torch.cuda.synchronize()
    for i in (0, 1):
        assert outs[i][0].cpu().double().item() == refs[i][0] and int(outs[i][1].item()) == refs[i][1]
    assert torch.cuda.mem_get_info()[0] == free0                       # the calls allocated nothing on the device
    # n_active may be NULL; an empty candidate list gives 0
    ctx2.tt_energy_static(probs[2], e)
    torch.cuda.synchronize()
    assert e.cpu().double().item() == refs[2][0]
    empty = ctx2.problem(probs[2][1][0], probs[2][1][1], torch.zeros((0, 2), dtype=torch.int32, device=DEV))
    ctx2.tt_energy_static(empty, e, na)
    torch.cuda.synchronize()
    assert e.item() == 0.0 and na.item() == 0
    ctx.close()
    ctx2.close()


def test_energy_static_rejects_sizes_beyond_the_static_array():
    from paper_2606_06511_b200 import tt
    ctx = tt.Context(torch.float64, 1, 1.0, 0)
    pos = torch.rand(30, 3, dtype=torch.float64, device=DEV)
    tris = torch.arange(30, dtype=torch.int32, device=DEV).reshape(10, 3).contiguous()
    n = tt.TT_STATIC_MAX_PAIRS + 1
    prs = torch.zeros((n, 2), dtype=torch.int32, device=DEV)
    prs[:, 1] = 1
    e = torch.full((1,), -1.0, dtype=torch.float64, device=DEV)
    with pytest.raises(tt.TTError) as ei:
        ctx.tt_energy_static(ctx.problem(pos, tris, prs), e)
    assert ei.value.status == TT_ERR_CAPACITY and "TT_STATIC_MAX_PAIRS" in str(ei.value)
    torch.cuda.synchronize()
    assert e.item() == -1.0                                            # nothing was launched
    # exactly the maximum is accepted (all candidates are the same separated pair or not: only the count matters here)
    ctx.tt_energy_static(ctx.problem(pos, tris, prs[:-1].contiguous()), e)
    torch.cuda.synchronize()
    ref = torch.zeros(1, dtype=torch.float64, device=DEV)
    ctx.tt_energy(ctx.problem(pos, tris, prs[:-1].contiguous()), ref)
    torch.cuda.synchronize()
    assert e.item() == ref.item()
    ctx.close()
