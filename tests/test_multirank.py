"""N > 1 path of bench.py on CPU: two gloo ranks, replicas only.

Every rank runs the same design independently; the only collectives are the barrier and the max-reduce of the per-rank
time, and `value` = N x units / max-over-ranks time.  This test drives exactly those helpers of bench.py with
world_size 2 over the gloo backend (rendezvous on 127.0.0.1), plus the reference arm's rank gating."""
import os
import socket
import subprocess
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
    local_ms = 100.0 + 50.0 * rank  # rank 1 is the slow replica
    dist.barrier()
    ms_max = bench.reduce_max(local_ms, "cpu")
    value = bench.whole_job_value(1.0e9, world, ms_max)
    out[rank] = (ms_max, value)
    dist.barrier()
    dist.destroy_process_group()


def test_two_gloo_ranks_take_the_slowest_replica():
    world, port = 2, _free_port()
    with mp.Manager() as mgr:
        out = mgr.dict()
        mp.spawn(_worker, args=(world, port, out), nprocs=world, join=True)
        res = dict(out)
    assert set(res) == {0, 1}
    for rank in (0, 1):
        ms_max, value = res[rank]
        assert ms_max == 150.0
        assert abs(value - 2 * 1.0e9 / 0.150) < 1e-3


def test_single_rank_needs_no_process_group():
    sys.path.insert(0, ROOT)
    import bench

    assert bench.reduce_max(12.5, "cpu") == 12.5
    assert bench.whole_job_value(10.0, 1, 1000.0) == 10.0


def test_reference_arm_runs_on_rank_zero_only():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1",
                        "--warmup", "0", "--config", "1"], env=env, capture_output=True, text=True, timeout=120)
    assert r.returncode == 0 and r.stdout.strip() == ""
