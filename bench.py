#!/usr/bin/env python
"""bench.py -- throughput of the whole hot path.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--pairs P] [--dtype f64|f32]

One "step" = one pass over all hot-path rows on one batch of synthetic input (BASELINE.json
configs[4], the throughput sweep: 2M-triangle random soup, P seeded candidate pairs, ~50 % active):
tt_hess_symbolic (classification a1/a2, compaction a2', BSR pattern a4) + tt_energy_grad_hess
(a3 + a4: energy, gradient, BSR values) + tt_hess_vec (a5).  Prints ONE JSON line on stdout.

  value        candidate pairs / s, inputs already resident in HBM (CUDA events on the launching stream)
  e2e          the same through tt_energy_grad_hess_host: pinned HOST buffers, H2D + D2H inside the timed region
  roofline     dominant kernel (k_assemble): algorithmic bytes / its CUDA-event duration vs measured HBM peak
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
    ap.add_argument("--pairs", type=int, default=10_000_000)
    ap.add_argument("--tris", type=int, default=2_000_000)
    ap.add_argument("--dtype", default="f64", choices=["f64", "f32"])
    ap.add_argument("--hess-mode", type=int, default=1)
    ap.add_argument("--broad-phase", default=None, choices=["config2", "config3"],
                    help="time tt_broad_phase (SURVEY 8(f) NEXT-1) on that mesh instead of the hot path; prints its own JSON line")
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


def make_problem(args, rank, device):
    from paper_2606_06511_b200 import inputs
    t = time.time()
    pb = inputs.config4_sweep(n_tris=args.tris, n_pairs=args.pairs, seed=rank_seed(inputs.BASE_SEED + 4, rank),
                              device=device)
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
            "sample": "first %d of %d candidate pairs of the same workload, energy+grad+BSR+H.p, %.1f s wall" % (n, pb.n_pairs, t)}


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


def main():
    args = parse()
    if args.impl == "reference":
        run_reference(args)
        return
    if args.broad_phase:
        run_broad_phase(args)
        return
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
    pos_np = pb.pos if args.dtype == "f64" else pb.pos.astype(np.float32)
    pos = torch.from_numpy(pos_np).to(dev)
    tris = torch.from_numpy(pb.tris).to(dev)
    pairs = torch.from_numpy(pb.pairs).to(dev)
    P, nV, nT = pb.n_pairs, pb.n_verts, pb.n_tris
    ctx = tt.Context(tdt, args.hess_mode, 1.0, local_rank)
    prob = ctx.problem(pos, tris, pairs)
    stream = torch.cuda.current_stream()

    # sizes are a property of the input: allocate outputs once (a Newton loop would do the same)
    nnzb, n_active = ctx.tt_hess_symbolic(prob)
    energy = torch.zeros(1, dtype=tdt, device=dev)
    grad = torch.empty((nV, 3), dtype=tdt, device=dev)
    rowptr = torch.empty(nV + 1, dtype=torch.int32, device=dev)
    colind = torch.empty(max(nnzb, 1), dtype=torch.int32, device=dev)
    vals = torch.empty((max(nnzb, 1), 3, 3), dtype=tdt, device=dev)
    pvec = torch.randn((nV, 3), dtype=tdt, device=dev)
    yvec = torch.empty_like(pvec)
    log("[bench] rank %d: A=%d nnzb=%d (vals %.2f GB)" % (rank, n_active, nnzb, nnzb * 9 * w / 1e9))

    phase_ev = []                                     # per timed step: 4 events around the three calls

    def step(record=False):
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(4)] if record else None
        if record:
            ev[0].record(stream)
        ctx.tt_hess_symbolic(prob)
        if record:
            ev[1].record(stream)
        ctx.tt_energy_grad_hess(prob, energy, grad, rowptr, colind, vals, max(nnzb, 1))
        if record:
            ev[2].record(stream)
        ctx.tt_hess_vec(prob, pvec, yvec)
        if record:
            ev[3].record(stream)
            phase_ev.append(ev)

    for _ in range(args.warmup):
        step()
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    sampler = ClockSampler(local_rank) if rank == 0 else None
    l0 = ctx.tt_stats()["launches"]
    kms = {"classify": [], "assemble": [], "hess_vec": []}
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    t_wall0 = time.time()
    ev0.record(stream)
    for _ in range(args.steps):
        step(record=True)
        for k, v in ctx.tt_kernel_ms().items():      # waits for the step's last kernel; no extra work
            kms[k].append(v)
    ev1.record(stream)
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    t_wall1 = time.time()
    launches = ctx.tt_stats()["launches"] - l0
    ms_total = ev0.elapsed_time(ev1)
    ms_total, P_all = aggregate_ranks(ms_total, P, world, dev)
    clocks = sampler.stop(t_wall0, t_wall1) if sampler else None
    ms_step = ms_total / args.steps
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
        del vals, colind                              # the host call keeps its own device BSR
        torch.cuda.empty_cache()

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
               "note": "tt_energy_grad_hess_host: pinned host pos/tris/pairs/p in; energy, grad, y out; BSR left on device"}

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel (k_assemble), DESIGN.md "Roofline" ----
    hbm, peak_src = peaks()
    n_touch = ctx.tt_stats()["n_touched_tris"]
    rows_touched = int((rowptr[1:] != rowptr[:-1]).sum().item())
    alg_bytes = 9 * w * nnzb + 3 * w * rows_touched + 12 * n_touch + 8 * n_active + 3 * w * 3 * n_touch
    asm_ms = float(np.mean(kms["assemble"]))
    achieved = alg_bytes / (asm_ms * 1e-3) / 1e9
    traffic = None
    tpath = os.path.join(ROOT, "profiles", "k_assemble_traffic.csv")   # ncu dram bytes per launch, same workload
    if os.path.exists(tpath):
        import csv
        with open(tpath) as f:
            for row in csv.DictReader(f):
                if int(row["pairs"]) == args.pairs and row["dtype"] == args.dtype:
                    traffic = int(row["dram_bytes_per_launch"])
    roofline = {"bound": "hbm", "kernel": "k_assemble", "achieved": achieved, "peak": hbm, "unit": "GB/s",
                "frac": achieved / hbm, "traffic": traffic, "peak_source": peak_src,
                "algorithmic_bytes_per_launch": int(alg_bytes), "kernel_ms": asm_ms,
                "share_of_step": asm_ms / ms_step}

    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        cpu = cpu_baseline(pb, args.hess_mode)

    out = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
           "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
           "dtype": args.dtype, "data": "synthetic",
           "config": {"workload": "BASELINE configs[4] throughput sweep: %d-triangle random soup, %d candidate pairs, "
                                  "%.1f%% active, energy+grad+BSR Hessian (+pattern) + one matrix-free H.p per step"
                                  % (nT, P, 100.0 * n_active / max(P, 1)),
                      "n_tris": nT, "n_verts": nV, "n_pairs": P, "n_active": n_active, "nnzb": nnzb,
                      "hess_mode": args.hess_mode, "replicas": world,
                      "l2": "inputs (%.0f MB) and outputs (%.1f GB) exceed the 126 MB L2; no flush needed" % (
                          (pos.numel() * w + tris.numel() * 4 + pairs.numel() * 4) / 1e6, nnzb * 9 * w / 1e9)},
           "roofline": roofline, "cpu_baseline": cpu, "e2e": e2e, "gpu_launches": int(launches),
           "clocks": clocks,
           "kernel_ms": {k: float(np.mean(v)) for k, v in kms.items()},
           "phase_ms": {name: float(np.mean([e[i].elapsed_time(e[i + 1]) for e in phase_ev]))
                        for i, name in enumerate(("tt_hess_symbolic", "tt_energy_grad_hess", "tt_hess_vec"))},
           "active_pairs_per_s": n_active * world / (ms_step * 1e-3)}
    print(json.dumps(out), flush=True)
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
