"""N > 1 host logic on CPU: two gloo ranks reduce their timings to the slowest rank's and the whole-job
rate counts both replicas (bench.py's multi-GPU leg; replicas only)."""
import os
import socket
import subprocess
import sys

import pytest

torch = pytest.importorskip("torch")

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, q):
    import torch.distributed as dist
    from paper_1509_07370_b200 import ranks
    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    dev_total, wall = ranks.max_over_ranks([0.010 * (rank + 1), 0.5 - 0.1 * rank])
    q.put((rank, dev_total, wall, ranks.whole_job_rate(1000, 4, dev_total, world)))
    dist.barrier()
    dist.destroy_process_group()


def test_max_over_two_gloo_ranks():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    got = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, dev_total, wall, rate in got:
        assert dev_total == pytest.approx(0.020)          # rank 1 is the slowest on the device
        assert wall == pytest.approx(0.5)                 # rank 0 is the slowest on the wall clock
        assert rate == pytest.approx(2 * 1000 * 4 / 0.020)


def test_single_process_is_identity():
    from paper_1509_07370_b200 import ranks
    assert ranks.max_over_ranks([1.5, 2.5]) == [1.5, 2.5]
    assert ranks.whole_job_rate(10, 2, 4.0, 1) == 5.0


def test_reference_arm_only_rank0_prints():
    """`bench.py --impl reference` under torchrun: ranks other than 0 exit 0 without work or output."""
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2"],
                       env=env, capture_output=True, text=True, timeout=120)
    assert r.returncode == 0 and r.stdout.strip() == ""
