"""N>1 path of bench.py on CPU (gloo, world_size 2): replicas only -- every rank gets its own seeded
batch, whole-job time is the MAX over ranks and whole-job pairs the SUM."""
import os
import socket
import sys

import pytest

torch = pytest.importorskip("torch")
import torch.multiprocessing as mp  # noqa: E402

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    import torch.distributed as dist
    import bench
    from paper_2606_06511_b200 import inputs
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    pb = inputs.config4_sweep(n_tris=2_000, n_pairs=5_000 + 1_000 * rank, seed=bench.rank_seed(inputs.BASE_SEED + 4, rank))
    ms, pairs = bench.aggregate_ranks(10.0 + 5.0 * rank, pb.n_pairs, world, "cpu")
    q.put((rank, ms, pairs, pb.n_pairs, int(pb.pairs[:64].sum())))
    dist.barrier()
    dist.destroy_process_group()


def test_two_replicas_gloo():
    world = 2
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (r0, ms0, n0, p0, h0), (r1, ms1, n1, p1, h1) = res
    assert ms0 == ms1 == 15.0                      # max over ranks
    assert n0 == n1 == float(p0 + p1)              # sum over ranks
    assert h0 != h1                                # different seeded batches


def test_single_rank_is_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.aggregate_ranks(3.5, 100, 1) == (3.5, 100.0)
