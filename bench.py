#!/usr/bin/env python
"""bench.py -- throughput of the whole hot path.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 0..4] [--pairs P]
                    [--dtype f64|f32] [--sweep P1,P2,...]

One "step" = one pass over all hot-path rows on one batch of synthetic input (BASELINE.json
configs[4], the throughput sweep: 2M-triangle random soup, P seeded candidate pairs, ~50 % active):
tt_hess_symbolic (classification a1/a2, compaction a2', BSR pattern a4) + tt_energy_grad_hess
(a3 + a4: energy, gradient, BSR values) + tt_hess_vec (a5).  Prints ONE JSON line on stdout.

  value        candidate pairs / s, inputs already resident in HBM (CUDA events on the launching stream)
  e2e          the same through tt_energy_grad_hess_host: pinned HOST buffers, H2D + D2H inside the timed region
  roofline     dominant kernel (k_assemble): algorithmic bytes / its CUDA-event duration vs measured HBM peak
  roofline_all the same for each of the three calls of the step, and step_frac for the step as a whole
  sweep        config 4 only: the same step at other points of BASELINE's 1M-50M sweep (fewer steps each)
  cpu_baseline the CPU oracle, as it stands, on a bounded sample (rank 0, N=1)

--impl reference times the oracle (the tier's reference arm).  N>1 (torchrun): independent
replicas, one per GPU, no collective on the data path ("replicas only").
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "tri-pairs/s for energy+grad+Hessian assembly (fp64), % of roofline"
UNIT = "pairs/s"


def log(*a):
    print(*a, file=sys.stderr, flush=True)


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=4, choices=[0, 1, 2, 3, 4],
                    help="BASELINE.json configs[i]; 4 (the throughput sweep the metric is quoted on) is the default")
    ap.add_argument("--pairs", type=int, default=10_000_000, help="config 4: candidate pairs of the headline workload")
    ap.add_argument("--sweep", default="1000000,50000000",
                    help="config 4: further sweep points reported under 'sweep' (comma separated pair counts, '' = none)")
    ap.add_argument("--sweep-steps", type=int, default=5)
    ap.add_argument("--tris", type=int, default=2_000_000)
    ap.add_argument("--dtype", default="f64", choices=["f64", "f32"])
    ap.add_argument("--hess-mode", type=int, default=1)
    ap.add_argument("--broad-phase", default=None, choices=["config2", "config3"],
                    help="time tt_broad_phase (SURVEY 8(f) NEXT-1) on that mesh instead of the hot path; prints its own JSON line")
    ap.add_argument("--solver", action="store_true",
                    help="time the consumer (SURVEY 8(f) NEXT-2) on the same workload instead of the hot path: tt_bsr_spmv "
                         "against its HBM roofline, tt_pcg_solve iterations/s (assembled and matrix-free); prints its own JSON line")
    ap.add_argument("--untangle", action="store_true",
                    help="run tt_untangle (broad phase + Newton step with line search, SURVEY 8(f) NEXT-2 / NEXT-4) on the mesh "
                         "given by --config (1, 2 or 3) for --steps steps; prints its own JSON line")
    ap.add_argument("--membrane", type=float, default=0.0,
                    help="with --untangle: stiffness k of the edge-spring membrane (SURVEY 8(f) NEXT-4, DESIGN.md A18); 0 = none")
    ap.add_argument("--k4-phases", action="store_true",
                    help="phase timers of the assembly kernel on the headline workload: needs the profiling build "
                         "(python -m paper_2606_06511_b200.build --profile); prints its own JSON line")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    return ap.parse_args()


def peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            d = json.load(f)
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index):
        self.rows = []
        self.proc = None
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(gpu_index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), line.strip()))

    def stop(self, t0, t1):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        sm, smax, reasons = [], [], set()
        for t, line in self.rows:
            f = [x.strip() for x in line.split(",")]
            if len(f) < 9:
                continue
            try:
                inside = t0 - 0.05 <= t <= t1 + 0.15
                if inside:
                    sm.append(float(f[1]))
                    smax.append(float(f[2]))
                    for name, val in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), f[5:9]):
                        if val.lower().startswith("active"):
                            reasons.add(name)
            except ValueError:
                continue
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(smax) if smax else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def aggregate_ranks(ms_local, pairs_local, world, device="cpu"):
    """Whole-job numbers of N independent replicas: time = MAX over ranks,
    pairs = SUM over ranks.  One all-reduce each, outside the timed region; backend-agnostic
    (nccl on the GPU box, gloo in tests/test_bench_ranks.py)."""
    if world <= 1:
        return float(ms_local), float(pairs_local)
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(ms_local)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    n = torch.tensor([float(pairs_local)], dtype=torch.float64, device=device)
    dist.all_reduce(n, op=dist.ReduceOp.SUM)
    return float(t.item()), float(n.item())


def rank_seed(base_seed, rank):
    """Every replica works on its own seeded batch."""
    return base_seed + 1000 * rank


def make_problem(args, rank, device, n_pairs=None):
    from paper_2606_06511_b200 import inputs
    t = time.time()
    if args.config == 4:
        pb = inputs.config4_sweep(n_tris=args.tris, n_pairs=n_pairs or args.pairs,
                                  seed=rank_seed(inputs.BASE_SEED + 4, rank), device=device)
    else:
        pb = inputs.by_name("config%d" % args.config, seed=rank_seed(inputs.BASE_SEED + args.config, rank))
    log("[bench] rank %d generated %s: nV=%d nT=%d P=%d in %.1fs" % (rank, pb.name, pb.n_verts, pb.n_tris, pb.n_pairs,
                                                                    time.time() - t))
    return pb


def oracle_step(oracle, pb, n_sample, hess_mode, p):
    """The oracle's whole hot path on the first n_sample candidate pairs (as it stands)."""
    prs = pb.pairs[:n_sample]
    t = time.perf_counter()
    r = oracle.assemble(pb.pos, pb.tris, prs, 1.0, hess_mode)
    oracle.hess_vec_pairs(pb.n_verts, pb.tris, prs, r["active"], r["tc"], r["J"], p, hess_mode)
    return time.perf_counter() - t


def cpu_baseline(pb, hess_mode, budget_s=15.0):
    import oracle
    oracle.build()
    rng = np.random.default_rng(0)
    p = rng.normal(size=pb.pos.shape)
    n0 = min(pb.n_pairs, 20_000)
    t0 = oracle_step(oracle, pb, n0, hess_mode, p)
    n = int(min(pb.n_pairs, max(n0, n0 * budget_s / max(t0, 1e-3))))
    t = oracle_step(oracle, pb, n, hess_mode, p)
    return {"value": n / t, "unit": UNIT, "cores": oracle.max_threads(), "kind": "oracle",
            "sample": "first %d of %d candidate pairs of the same workload, energy+grad+BSR+H.p, %.1f s wall" % (n, pb.n_pairs, t),
            "note": "the oracle as it stands: per-pair loop (18-partial dual numbers) and H.p run under OpenMP on `cores` "
                    "threads, its pattern sort and BSR accumulation are serial; a baseline, not a tuned CPU figure"}


def run_reference(args):
    """--impl reference: the oracle timed on the host cores, rank 0 only."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle
    oracle.build()
    from paper_2606_06511_b200 import inputs
    n_pairs = min(args.pairs, 1_000_000)      # the oracle only ever sees a bounded sample
    pb = inputs.config4_sweep(n_tris=args.tris, n_pairs=n_pairs, seed=inputs.BASE_SEED + 4)
    p = np.random.default_rng(0).normal(size=pb.pos.shape)
    t0 = oracle_step(oracle, pb, 20_000, args.hess_mode, p)
    budget = 120.0 / max(args.steps + args.warmup, 1)
    n = int(min(pb.n_pairs, max(20_000, 20_000 * budget / max(t0, 1e-3))))
    for _ in range(args.warmup):
        oracle_step(oracle, pb, n, args.hess_mode, p)
    ts = [oracle_step(oracle, pb, n, args.hess_mode, p) for _ in range(args.steps)]
    tot = sum(ts)
    val = n * args.steps / tot
    sample = "first %d candidate pairs per step of config4 sweep (nT=%d), energy+grad+BSR+H.p" % (n, args.tris)
    out = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
           "warmup": args.warmup, "ms_per_step": 1e3 * tot / args.steps, "higher_is_better": True, "scaling": "weak",
           "vs_baseline": None, "dtype": "f64", "data": "synthetic",
           "config": {"workload": "config4 sweep: %d-tri soup, %d pairs, ~50%% active (oracle sample %d pairs/step)" % (args.tris, args.pairs, n)},
           "cpu_baseline": {"value": val, "unit": UNIT, "cores": oracle.max_threads(), "kind": "oracle", "sample": sample},
           "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
           "gpu_launches": 0}
    print(json.dumps(out), flush=True)


def run_broad_phase(args):
    """Side measurement, not the headline: tt_broad_phase on a mesh config (inputs resident, CUDA events)."""
    import torch
    from paper_2606_06511_b200 import inputs, tt
    dev = torch.device("cuda", 0)
    if args.broad_phase == "config2":
        pb, inflate = inputs.config2_cloth(), 0.002
        pos_np, tris_np = pb.pos, pb.tris
    else:   # the torus mesh without the generator's own (CPU) candidate search
        saved = inputs.aabb_candidates
        inputs.aabb_candidates = lambda pos, tris, inflate=0.0, max_pairs=None: np.zeros((0, 2), dtype=np.int32)
        try:
            pb = inputs.config3_torus()
        finally:
            inputs.aabb_candidates = saved
        pos_np, tris_np, inflate = pb.pos, pb.tris, 0.0
    ctx = tt.Context(torch.float64, 1, 1.0, 0)
    pos = torch.from_numpy(pos_np).to(dev)
    tris = torch.from_numpy(tris_np).to(dev)
    stream = torch.cuda.current_stream()
    for _ in range(args.warmup):
        out = ctx.tt_broad_phase(pos, tris, inflate)
    torch.cuda.synchronize()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ev0.record(stream)
    for _ in range(args.steps):
        out = ctx.tt_broad_phase(pos, tris, inflate)
    ev1.record(stream)
    torch.cuda.synchronize()
    ms = ev0.elapsed_time(ev1) / args.steps
    n = int(out.shape[0])
    print(json.dumps({"metric": "broad phase: candidate pairs/s (tt_broad_phase, fp64 boxes)", "value": n / (ms * 1e-3),
                      "unit": UNIT, "n_gpus": 1, "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms,
                      "higher_is_better": True, "dtype": "f64", "data": "synthetic",
                      "config": {"workload": "%s mesh, %d triangles, inflate %g -> %d candidate pairs" % (
                          args.broad_phase, tris_np.shape[0], inflate, n)}}), flush=True)
    ctx.close()


def run_solver(args):
    """Side measurement, not the headline: the consumer of the assembly on config 4 (or --config), inputs resident, CUDA events."""
    import torch
    from paper_2606_06511_b200 import tt
    dev = torch.device("cuda", 0)
    tdt = torch.float64 if args.dtype == "f64" else torch.float32
    w = 8 if args.dtype == "f64" else 4
    pb = make_problem(args, 0, "cuda:0")
    ctx = tt.Context(tdt, 2, 1.0, 0)     # PSD2: H + mu I is SPD
    pos_np = pb.pos if w == 8 else pb.pos.astype(np.float32)
    out = tt.assemble(ctx, torch.from_numpy(pos_np).to(dev), torch.from_numpy(pb.tris).to(dev), torch.from_numpy(pb.pairs).to(dev))
    nV, nnzb = pb.n_verts, out["nnzb"]
    x = torch.randn((nV, 3), dtype=tdt, device=dev)
    y = torch.empty_like(x)
    stream = torch.cuda.current_stream()
    hbm, peak_src = peaks()

    def timed(fn, reps):
        for _ in range(args.warmup):
            fn()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for _ in range(reps):
            fn()
        e1.record(stream)
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) / reps

    ms_spmv = timed(lambda: ctx.tt_bsr_spmv(out["rowptr"], out["colind"], out["vals"], x, y, 0.0), args.steps)
    b_spmv = (9 * w + 4) * nnzb + 4 * (nV + 1) + 6 * w * nV          # values + colind, rowptr, x gathered once + y
    diag = out["vals"][out["colind"] == torch.repeat_interleave(torch.arange(nV, device=dev), (out["rowptr"][1:] - out["rowptr"][:-1]).long())]
    mu = float(diag.double().diagonal(dim1=1, dim2=2).sum(1).mean().item()) / 3 * 1e-2     # 1 % of the mean diagonal
    minv = torch.empty((nV, 3, 3), dtype=tdt, device=dev)
    ms_jac = timed(lambda: ctx.tt_block_jacobi(out["rowptr"], out["colind"], out["vals"], minv, mu), args.steps)
    iters = 20
    ms_pcg = timed(lambda: ctx.tt_pcg_solve(out["prob"], out["grad"], y, rowptr=out["rowptr"], colind=out["colind"], vals=out["vals"],
                                            minv=minv, max_iter=iters, rtol=0.0, shift=mu, want_stats=False), max(2, args.steps // 4))
    ms_pcg_mf = timed(lambda: ctx.tt_pcg_solve(out["prob"], out["grad"], y, max_iter=iters, rtol=0.0, shift=mu, want_stats=False),
                      max(2, args.steps // 4))
    print(json.dumps({"metric": "consumer: tt_bsr_spmv GB/s against the HBM roofline; tt_pcg_solve iterations/s", "n_gpus": 1,
                      "dtype": args.dtype, "data": "synthetic", "steps": args.steps, "warmup": args.warmup,
                      "config": {"workload": "BASELINE %s: %d triangles, %d candidate pairs, nnzb %d, PSD2 Hessian, shift %.3g" % (
                          WORKLOADS[args.config], pb.n_tris, pb.n_pairs, nnzb, mu)},
                      "spmv": {"ms": ms_spmv, "algorithmic_bytes": int(b_spmv), "achieved": b_spmv / (ms_spmv * 1e-3) / 1e9, "peak": hbm,
                               "unit": "GB/s", "frac": b_spmv / (ms_spmv * 1e-3) / 1e9 / hbm, "peak_source": peak_src, "bound": "hbm"},
                      "block_jacobi_ms": ms_jac,
                      "pcg_assembled": {"iters": iters, "ms_per_solve": ms_pcg, "iters_per_s": iters / (ms_pcg * 1e-3)},
                      "pcg_matrix_free": {"iters": iters, "ms_per_solve": ms_pcg_mf, "iters_per_s": iters / (ms_pcg_mf * 1e-3)}}), flush=True)
    ctx.close()


def run_k4_phases(args):
    """Diagnostic, not a bench value: where a round of k_assemble_tile spends its cycles.  Loads the profiling build
    (-DTT_K4_PROFILE: clock64() marks summed per phase over every round of a launch, read through tt_debug_k4_prof);
    the marks serialise the phases a little, so the kernel runs a few per cent slower than the product's."""
    import ctypes
    from paper_2606_06511_b200 import build as _b
    os.environ["TT_LIB_PATH"] = str(_b.build_profile())
    import torch
    from paper_2606_06511_b200 import inputs, tt
    dev = torch.device("cuda", 0)
    pb = inputs.config4_sweep(n_tris=args.tris, n_pairs=args.pairs)
    tdt = torch.float64 if args.dtype == "f64" else torch.float32
    ctx = tt.Context(tdt, args.hess_mode, 1.0, 0)
    pos = torch.from_numpy(pb.pos).to(dev).to(tdt).contiguous()
    out = tt.assemble(ctx, pos, torch.from_numpy(pb.tris).to(dev), torch.from_numpy(pb.pairs).to(dev), want_hess=True)
    torch.cuda.synchronize()
    buf = (ctypes.c_ulonglong * 16)()
    ctx.lib.tt_debug_k4_prof(buf, 1)
    n = max(int(args.steps), 1)
    for _ in range(n):
        ctx.tt_energy_grad_hess(out["prob"], out["energy"], out["grad"], out["rowptr"], out["colind"], out["vals"], out["nnzb"])
    torch.cuda.synchronize()
    ms = ctx.tt_kernel_ms()["assemble"]
    ctx.lib.tt_debug_k4_prof(buf, 0)
    names = ["derivatives (eval_core)", "operand loads, wait for the copy engine, unpermute", "slot offsets, diagonal factors",
             "staging + barrier", "per-triangle sums + barrier", "rows: waits, offsets, off-diagonal blocks",
             "rows: diagonal blocks, next positions", "rows: proxy fence, barrier, bulk-copy issue", "energy, loop"]
    v = [float(buf[i]) for i in range(9)]
    tot = sum(v) or 1.0
    st = ctx.tt_stats()
    print(json.dumps({"metric": "k_assemble_tile phase timers (profiling build, -DTT_K4_PROFILE)", "n_gpus": 1, "dtype": args.dtype,
                      "data": "synthetic", "config": {"workload": "BASELINE %s: %d triangles, %d candidate pairs" % (WORKLOADS[4], pb.n_tris, pb.n_pairs)},
                      "launches": n, "kernel_ms_profiling_build": ms, "rounds": st["rounds"],
                      "cycles_per_round_per_warp": tot / n / max(st["rounds"], 1),
                      "share": {nm: x / tot for nm, x in zip(names, v)}}), flush=True)
    ctx.close()


def run_untangle(args):
    """Side measurement, not the headline: the untangling loop on a mesh config -- per step one tt_broad_phase, one symbolic +
    numeric call, a block-Jacobi PCG solve and the Armijo line search on tt_energy.  Wall time per step (the loop synchronises
    once per trial step length), energy and active-pair count along the way."""
    import torch
    from paper_2606_06511_b200 import inputs, tt
    dev = torch.device("cuda", 0)
    cfg = args.config if args.config in (1, 2, 3) else 1
    pb = inputs.by_name("config%d" % cfg)
    inflate = {1: 0.02, 2: 0.002, 3: 0.0}[cfg]
    ctx = tt.Context(torch.float64, 2, 1.0, 0)     # PSD2
    tris = torch.from_numpy(pb.tris).to(dev)
    mu, iters = 1e-3, 30
    mbk = float(args.membrane)
    kw = dict(inflate=inflate, mu=mu, pcg_iter=iters, membrane=mbk > 0.0, matrix_free=mbk > 0.0)
    rest = torch.from_numpy(pb.pos).to(dev)
    if mbk > 0.0:
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        ctx.tt_membrane_build(rest, tris, mbk)
        torch.cuda.synchronize()
        ms_build = 1e3 * (time.perf_counter() - t0)
    pos = rest.clone()
    ctx.tt_untangle(pos, tris, max_steps=2, **kw)       # warm-up (workspace allocation)
    pos = rest.clone()
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    hist = ctx.tt_untangle(pos, tris, max_steps=args.steps, **kw)
    torch.cuda.synchronize()
    dt = time.perf_counter() - t0
    disp = float((pos - rest).norm(dim=1).max())
    t64 = tris.long()
    ed = torch.cat([t64[:, [0, 1]], t64[:, [1, 2]], t64[:, [2, 0]]])
    strain = float(((pos[ed[:, 0]] - pos[ed[:, 1]]).norm(dim=1) / (rest[ed[:, 0]] - rest[ed[:, 1]]).norm(dim=1) - 1).abs().max())
    print(json.dumps({"metric": "untangling loop (tt_untangle): ms per step, energy and active pairs along the way", "n_gpus": 1,
                      "dtype": "f64", "data": "synthetic", "steps": len(hist),
                      "config": {"workload": "BASELINE %s: %d triangles; inflate %g, PSD2, mu %g, %d PCG steps per Newton step" % (
                          WORKLOADS[cfg], pb.n_tris, inflate, mu, iters)},
                      "ms_per_step": 1e3 * dt / max(len(hist), 1), "all_accepted": all(h["accepted"] for h in hist),
                      "n_pairs": [hist[0]["n_pairs"], hist[-1]["n_pairs"]], "n_active": [h["n_active"] for h in hist][::max(1, len(hist) // 10)],
                      "energy": [hist[0]["energy0"]] + [h["energy1"] for h in hist][::max(1, len(hist) // 10)],
                      "max_vertex_displacement": disp, "max_edge_strain": strain,
                      "membrane": ({"stiffness": mbk, "build_ms": ms_build, "energy_membrane": hist[-1]["energy_membrane"],
                                    "back_end": "matrix-free, membrane block-Jacobi"} if mbk > 0.0 else None)}), flush=True)
    ctx.close()


WORKLOADS = {0: "configs[0] 64-triangle soup, all pairs", 1: "configs[1] two icospheres, inflated-AABB candidates",
             2: "configs[2] folded cloth 256x256, inflated-AABB candidates", 3: "configs[3] twisted torus 1M triangles, AABB candidates",
             4: "configs[4] throughput sweep: random soup, seeded random candidate pairs"}


def measure(ctx, pb, args, dev, steps, warmup, world=1, rank=0, sampler_rank0=False):
    """W warm-up + K timed steps of symbolic + numeric + H.p on one resident workload.  No synchronisation
    inside the timed loop: phase events are recorded on the launching stream, the library records the
    events of its three large kernels itself (tt_kernel_ms_mean), all read after the loop."""
    import torch
    import torch.distributed as dist
    tdt = ctx.dtype
    w = 8 if tdt == torch.float64 else 4
    pos_np = pb.pos if w == 8 else pb.pos.astype(np.float32)
    pos = torch.from_numpy(pos_np).to(dev)
    tris = torch.from_numpy(pb.tris).to(dev)
    pairs = torch.from_numpy(pb.pairs).to(dev)
    P, nV, nT = pb.n_pairs, pb.n_verts, pb.n_tris
    prob = ctx.problem(pos, tris, pairs)
    stream = torch.cuda.current_stream()
    # sizes are a property of the input: allocate outputs once (a Newton loop would do the same)
    nnzb, n_active = ctx.tt_hess_symbolic(prob)
    energy = torch.zeros(1, dtype=tdt, device=dev)
    grad = torch.empty((nV, 3), dtype=tdt, device=dev)
    # the BSR pattern stays where tt_hess_symbolic builds it (ctx-owned views, tt_hess_pattern): the numeric call
    # then writes the values only and does not duplicate rowptr / colind into a second pair of arrays
    rowptr, colind, _ = ctx.tt_hess_pattern(nV)
    vals = torch.empty((max(nnzb, 1), 3, 3), dtype=tdt, device=dev)
    pvec = torch.randn((nV, 3), dtype=tdt, device=dev)
    yvec = torch.empty_like(pvec)
    log("[bench] rank %d: P=%d A=%d nnzb=%d (vals %.2f GB)" % (rank, P, n_active, nnzb, nnzb * 9 * w / 1e9))
    phase_ev = []

    def step(record=False):
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(4)] if record else None
        if record:
            ev[0].record(stream)
        ctx.tt_hess_symbolic(prob)
        if record:
            ev[1].record(stream)
        rp_addr, ci_addr, _ = ctx.tt_hess_pattern_ptrs()   # re-read: a symbolic call may re-allocate its workspace
        ctx.tt_energy_grad_hess(prob, energy, grad, rp_addr, ci_addr, vals, max(nnzb, 1))
        if record:
            ev[2].record(stream)
        ctx.tt_hess_vec(prob, pvec, yvec)
        if record:
            ev[3].record(stream)
            phase_ev.append(ev)

    for _ in range(warmup):
        step()
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    ctx.tt_kernel_ms_mean(reset=True)
    sampler = ClockSampler(dev.index) if sampler_rank0 else None
    l0 = ctx.tt_stats()["launches"]
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    t_wall0 = time.time()
    ev0.record(stream)
    for _ in range(steps):
        step(record=True)
    ev1.record(stream)
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    t_wall1 = time.time()
    launches = ctx.tt_stats()["launches"] - l0
    kms, kcount = ctx.tt_kernel_ms_mean(reset=True)          # events of the timed steps only (ring of 64 launches)
    ms_local = ev0.elapsed_time(ev1)
    ms_total, P_all = aggregate_ranks(ms_local, P, world, dev)
    clocks = sampler.stop(t_wall0, t_wall1) if sampler else None
    ms_step = ms_total / steps
    phase_ms = {name: float(np.mean([e[i].elapsed_time(e[i + 1]) for e in phase_ev]))
                for i, name in enumerate(("tt_hess_symbolic", "tt_energy_grad_hess", "tt_hess_vec"))}

    # ---- algorithmic bytes (every unique item once; staging is not counted) ----
    hbm, peak_src = peaks()
    st = ctx.tt_stats()
    n_touch = st["n_touched_tris"]                                    # triangles of ACTIVE pairs
    rowptr, colind, _ = ctx.tt_hess_pattern(nV)                       # the views of the LAST symbolic call
    rows_touched = int((rowptr[1:] != rowptr[:-1]).sum().item())      # their vertices (= non-empty rows)
    cand_tris = int(torch.unique(pairs).numel())                      # triangles any CANDIDATE refers to
    cand_verts = int(torch.unique(tris[torch.unique(pairs).long()]).numel()) if P else 0
    b_sym = 8 * P + 12 * cand_tris + 3 * w * cand_verts + P // 8 + 4 * (nV + 1) + 4 * nnzb
    b_k4 = 9 * w * nnzb + 3 * w * rows_touched + 12 * n_touch + 8 * n_active + 3 * w * rows_touched
    b_num = b_k4 + 3 * w * nV                                         # + the dense gradient [nV,3]
    b_hv = 4 * n_active + 12 * n_touch + 3 * w * rows_touched + 6 * w * nV
    b_k1 = 8 * P + 12 * cand_tris + 3 * w * cand_verts + P // 8

    def roof(name, nbytes, ms):
        a = nbytes / (ms * 1e-3) / 1e9 if ms and ms > 0 else 0.0
        return {"call": name, "bound": "hbm", "algorithmic_bytes": int(nbytes), "ms": ms, "achieved": a, "peak": hbm,
                "unit": "GB/s", "frac": a / hbm}

    roofline_all = [roof("tt_hess_symbolic", b_sym, phase_ms["tt_hess_symbolic"]),
                    roof("tt_energy_grad_hess", b_num, phase_ms["tt_energy_grad_hess"]),
                    roof("tt_hess_vec", b_hv, phase_ms["tt_hess_vec"])]
    step_bytes = b_sym + b_num + b_hv
    res = dict(ms_step=ms_step, P_all=P_all, P=P, nV=nV, nT=nT, nnzb=nnzb, n_active=n_active, launches=int(launches),
               kernel_ms=kms, kernel_launches=kcount, phase_ms=phase_ms, clocks=clocks, roofline_all=roofline_all,
               step_frac=step_bytes / (ms_step * 1e-3) / 1e9 / hbm, step_bytes=int(step_bytes),
               k4=roof("k_assemble", b_k4, kms["assemble"]), k1=roof("k_classify", b_k1, kms["classify"]),
               k6=roof("k_entry_pipe", b_hv - 6 * w * nV + 3 * w * nV, kms["hess_vec"]),
               hbm=hbm, peak_src=peak_src, w=w, in_bytes=pos.numel() * w + tris.numel() * 4 + pairs.numel() * 4,
               tensors=(pos_np, pvec))
    del vals, colind, grad, rowptr, yvec
    torch.cuda.empty_cache()
    return res


def stored_traffic(kernel, pairs, dtype, config):
    """ncu dram__bytes_read.sum + dram__bytes_write.sum per launch, from the committed captures."""
    tpath = os.path.join(ROOT, "profiles", "k_assemble_traffic.csv")
    if not os.path.exists(tpath):
        return None, None
    import csv
    with open(tpath) as f:
        for row in csv.DictReader(f):
            if (row.get("kernel", "k_assemble") == kernel and int(row["pairs"]) == pairs and row["dtype"] == dtype
                    and int(row.get("config", 4)) == config):
                return int(row["dram_bytes_per_launch"]), row.get("capture", "profiles/")
    return None, None


def self_spawn(args):
    """`python bench.py --gpus N` without torchrun: start the N ranks ourselves (replicas only)."""
    import socket
    with socket.socket() as so:
        so.bind(("127.0.0.1", 0))
        port = so.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(args.gpus),
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    raise SystemExit(subprocess.call(cmd))


def main():
    args = parse()
    if args.impl == "reference":
        run_reference(args)
        return
    if args.broad_phase:
        run_broad_phase(args)
        return
    if args.solver:
        run_solver(args)
        return
    if args.k4_phases:
        run_k4_phases(args)
        return
    if args.untangle:
        run_untangle(args)
        return
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        self_spawn(args)
    import torch
    import torch.distributed as dist
    from paper_2606_06511_b200 import tt

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    tdt = torch.float64 if args.dtype == "f64" else torch.float32
    w = 8 if args.dtype == "f64" else 4
    pb = make_problem(args, rank, "cuda:%d" % local_rank)
    ctx = tt.Context(tdt, args.hess_mode, 1.0, local_rank)
    m = measure(ctx, pb, args, dev, args.steps, args.warmup, world, rank, sampler_rank0=(rank == 0))
    pos_np, pvec = m.pop("tensors")
    P, nV, nT, nnzb, n_active = m["P"], m["nV"], m["nT"], m["nnzb"], m["n_active"]
    ms_step, P_all = m["ms_step"], m["P_all"]
    value = P_all / (ms_step * 1e-3)

    # ---- e2e through the host-buffer C-ABI call (pinned host memory, copies inside the timed region) ----
    e2e = None
    if not args.no_e2e:
        pos_h = torch.from_numpy(pos_np).pin_memory()
        tris_h = torch.from_numpy(pb.tris).pin_memory()
        pairs_h = torch.from_numpy(pb.pairs).pin_memory()
        e_h = torch.zeros(1, dtype=tdt).pin_memory()
        g_h = torch.zeros((nV, 3), dtype=tdt).pin_memory()
        p_h = pvec.cpu().pin_memory()
        y_h = torch.zeros((nV, 3), dtype=tdt).pin_memory()

        def host_step():
            return ctx.tt_energy_grad_hess_host(pos_h, tris_h, pairs_h, e_h, g_h, None, None, None, 0, p_h, y_h)

        for _ in range(max(1, min(args.warmup, 2))):
            host_step()
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        k2 = max(1, min(args.steps, 5))
        t0 = time.perf_counter()
        for _ in range(k2):
            host_step()                               # synchronises the stream before returning
        t_e2e = (time.perf_counter() - t0) / k2
        if world > 1:
            tm = torch.tensor([t_e2e], dtype=torch.float64, device=dev)
            dist.all_reduce(tm, op=dist.ReduceOp.MAX)
            t_e2e = float(tm.item())
        h2d = pos_h.numel() * w + tris_h.numel() * 4 + pairs_h.numel() * 4 + p_h.numel() * w
        d2h = w + g_h.numel() * w + y_h.numel() * w
        e2e = {"value": P_all / t_e2e, "unit": UNIT, "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h),
               "ms_per_step": 1e3 * t_e2e, "steps": k2,
               "note": "tt_energy_grad_hess_host: pinned host pos/tris/pairs/p in; energy, grad, y out; the BSR "
                       "(%.2f GB) stays on the device for the PCG that consumes it there (tt_bsr_device / tt_pcg_solve); "
                       "copying it out too would add %.0f ms at ~55 GB/s PCIe Gen5" % (
                           nnzb * (9 * w + 4) / 1e9, nnzb * (9 * w + 4) / 55e9 * 1e3)}
        del pos_h, tris_h, pairs_h, g_h, p_h, y_h
    del pvec

    # ---- further points of the 1M-50M sweep (config 4, rank 0's replica only; fewer steps) ----
    sweep = None
    if args.config == 4 and args.sweep and world == 1:
        sweep = []
        ctx.close()
        torch.cuda.empty_cache()
        for n_pairs in [int(x) for x in args.sweep.split(",") if x]:
            if n_pairs == args.pairs:
                continue
            pbs = make_problem(args, rank, "cuda:%d" % local_rank, n_pairs)
            cs = tt.Context(tdt, args.hess_mode, 1.0, local_rank)
            ms = measure(cs, pbs, args, dev, args.sweep_steps, 3)
            ms.pop("tensors")
            sweep.append({"pairs": ms["P"], "n_active": ms["n_active"], "nnzb": ms["nnzb"], "steps": args.sweep_steps,
                          "ms_per_step": ms["ms_step"], "pairs_per_s": ms["P"] / (ms["ms_step"] * 1e-3),
                          "k4_ms": ms["k4"]["ms"], "k4_frac": ms["k4"]["frac"], "step_frac": ms["step_frac"],
                          "phase_ms": ms["phase_ms"], "kernel_ms": ms["kernel_ms"]})
            cs.close()
            del pbs
            torch.cuda.empty_cache()

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel: K4 (assembly) on the sweep; on the mesh configs
    #      (< 1 % of the candidates active) the step is the classification kernel K1 ----
    dom = m["k4"] if args.config == 4 else m["k1"]
    traffic, capture = stored_traffic(dom["call"], args.pairs if args.config == 4 else P, args.dtype, args.config)
    roofline = {"bound": "hbm", "kernel": dom["call"], "achieved": dom["achieved"], "peak": m["hbm"], "unit": "GB/s",
                "frac": dom["frac"], "traffic": traffic,
                "traffic_source": ("stored ncu capture (%s), not measured in this run" % capture) if traffic else None,
                "peak_source": m["peak_src"], "algorithmic_bytes_per_launch": dom["algorithmic_bytes"],
                "kernel_ms": dom["ms"], "share_of_step": dom["ms"] / ms_step,
                "kernel_launches_averaged": m["kernel_launches"]}

    # ---- what random gathers can reach on this memory system (tt_probe_gather), beside the copy bandwidth: K1 gathers
    #      6 vertices per candidate, K6 3 partner vertices + 3 partner p per directed entry ----
    gather = None
    try:
        gp = tt.tt_probe_gather(local_rank)
        k1_useful = 6 * 3 * w * P                      # bytes of vertex data K1 gathers (ids and pair list not counted)
        k6_useful = 2 * 3 * 3 * w * 2 * n_active       # partner positions + partner p per directed entry
        gather = {"vertex_items_gbs": gp["vertex_gbs"], "triangle_items_gbs": gp["triangle_gbs"], "unit": "GB/s of useful bytes",
                  "what": "random 24-byte / 72-byte fp64 items from a 144 MB array, one per thread (tt_probe_gather)",
                  "k_classify": {"useful_gather_bytes": int(k1_useful), "achieved_gbs": k1_useful / (m["kernel_ms"]["classify"] * 1e-3) / 1e9,
                                 "frac_of_vertex_gather": k1_useful / (m["kernel_ms"]["classify"] * 1e-3) / 1e9 / gp["vertex_gbs"]},
                  "k_entry_pipe": {"useful_gather_bytes": int(k6_useful), "achieved_gbs": k6_useful / (m["kernel_ms"]["hess_vec"] * 1e-3) / 1e9,
                                   "frac_of_triangle_gather": k6_useful / (m["kernel_ms"]["hess_vec"] * 1e-3) / 1e9 / gp["triangle_gbs"]}}
    except Exception as e:   # diagnostic only
        gather = {"error": str(e)}

    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        cpu = cpu_baseline(pb, args.hess_mode)

    out = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
           "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
           "dtype": args.dtype, "data": "synthetic",
           "config": {"workload": "BASELINE %s: %d triangles, %d candidate pairs, %.1f%% active; step = pattern "
                                  "(tt_hess_symbolic) + energy+grad+BSR Hessian (tt_energy_grad_hess) + one matrix-free H.p "
                                  "(tt_hess_vec)" % (WORKLOADS[args.config], nT, P, 100.0 * n_active / max(P, 1)),
                      "config_index": args.config, "n_tris": nT, "n_verts": nV, "n_pairs": P, "n_active": n_active,
                      "nnzb": nnzb, "hess_mode": args.hess_mode, "replicas": world,
                      "l2": ("inputs (%.0f MB) and outputs (%.1f GB) exceed the 126 MB L2; no flush needed" % (
                          m["in_bytes"] / 1e6, nnzb * 9 * w / 1e9)) if m["in_bytes"] + nnzb * 9 * w > 2.0e8 else
                            "working set fits the L2: every step rewrites the same buffers (L2-resident numbers, stated)"},
           "roofline": roofline, "roofline_all": m["roofline_all"], "step_frac": m["step_frac"],
           "step_algorithmic_bytes": m["step_bytes"],
           "cpu_baseline": cpu, "e2e": e2e, "gpu_launches": m["launches"],
           "clocks": m["clocks"], "kernel_ms": m["kernel_ms"],
           "kernel_roofline": {k: {"frac": m[k]["frac"], "algorithmic_bytes": m[k]["algorithmic_bytes"]} for k in ("k1", "k4", "k6")},
           "phase_ms": m["phase_ms"], "sweep": sweep, "gather_probe": gather,
           "active_pairs_per_s": n_active * world / (ms_step * 1e-3)}
    print(json.dumps(out), flush=True)
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
