"""The N > 1 path of bench.py is "replicas only": no data-path collective, just
a barrier and a MAX-over-ranks of the timings.  Covered here with world_size-2 gloo on CPU."""
import os
import socket
import subprocess
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, world: int, port: int, q):
    sys.path.insert(0, ROOT)
    import bench

    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    dist.barrier()
    # rank r "measured" (100 + 7 r) us per step and 250 - 3 r us end to end
    got = bench.max_over_ranks([100.0 + 7 * rank, 250.0 - 3 * rank], dist, torch.device("cpu"))
    dist.barrier()
    q.put((rank, got, bench.whole_job_tokens_per_s(world, 12, got[0])))
    dist.destroy_process_group()


def test_max_over_ranks_and_whole_job_value_world_size_2():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, got, tps in res:
        assert got == [107.0, 250.0]  # the slowest rank's time, on every rank
        assert abs(tps - 2 * 12 / 107e-6) < 1e-6  # all ranks' tokens over the slowest rank's step


def test_identity_without_process_group():
    sys.path.insert(0, ROOT)
    import bench

    assert bench.max_over_ranks([1.5, 2.5], None, torch.device("cpu")) == [1.5, 2.5]


def test_reference_arm_other_ranks_exit_without_work():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1",
                        "--warmup", "1"], env=env, capture_output=True, text=True, timeout=120)
    assert r.returncode == 0 and r.stdout.strip() == ""
