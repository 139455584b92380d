"""N > 1 path of bench.py on CPU (gloo, world_size 2): the path does not shard (replicas only), so the only
multi-rank logic is the max-over-ranks timing and the whole-job aggregate, plus the reference arm running on rank 0 alone."""
import os
import socket
import sys

import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    import bench
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ms, value = bench.aggregate(10.0 * (rank + 1), zones=1000, steps=4, world=world, device="cpu")
    out.put((rank, ms, value))
    dist.barrier()
    dist.destroy_process_group()


def test_replica_aggregate_takes_the_max_over_ranks():
    world = 2
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, out)) for r in range(world)]
    for p in procs:
        p.start()
    got = sorted(out.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=120)
        assert p.exitcode == 0
    for rank, ms, value in got:
        assert ms == 20.0                                   # the slower rank's time on every rank
        assert value == world * 1000 * 4 / 20e-3            # whole-job zone-cycles/s of both replicas


def test_reference_arm_runs_on_rank_zero_only(monkeypatch, capsys):
    sys.path.insert(0, ROOT)
    import bench
    monkeypatch.setenv("RANK", "1")
    monkeypatch.setenv("WORLD_SIZE", "2")

    class A:
        gpus, steps, warmup, n, workload = 2, 1, 0, 256, "cfg4"
    bench.run_reference(A)
    assert capsys.readouterr().out == ""
