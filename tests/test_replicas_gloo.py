"""N > 1 host logic on CPU (world_size 2, gloo, 127.0.0.1).  The path does not shard (replicas
only), so what there is to cover is bench.py's cross-rank bookkeeping: the max-over-ranks step time, the whole-job
value, and the reference arm printing on rank 0 only."""
import json
import os
import socket
import subprocess
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, q):
    import bench
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ms_local = 4.0 + 1.5 * rank  # rank 1 is the slow replica
    dist.barrier()
    ms = bench.max_over_ranks(ms_local, world, "cpu")
    q.put((rank, ms, bench.whole_job_value(world, 512 ** 3, ms)))
    dist.barrier()
    dist.destroy_process_group()


def test_replica_timing_is_the_max_over_ranks_and_value_is_the_whole_job():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    got = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, ms, value in got:
        assert ms == 5.5  # every rank sees the slowest replica's time
        assert abs(value - 2 * 512 ** 3 * 4 / 5.5e-3 / 1e9) < 1e-9  # two replicas' cell-stages over that time
    import bench
    assert bench.max_over_ranks(3.25, 1, "cpu") == 3.25  # N = 1: no collective


def test_reference_arm_prints_on_rank_0_only():
    env = dict(os.environ, WORLD_SIZE="2", MASTER_ADDR="127.0.0.1", MASTER_PORT=str(_free_port()), OMP_NUM_THREADS="2")
    cmd = [sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--workload", "C1",
           "--steps", "1", "--warmup", "1"]
    r1 = subprocess.run(cmd, env=dict(env, RANK="1", LOCAL_RANK="1"), capture_output=True, text=True, timeout=300)
    assert r1.returncode == 0 and r1.stdout.strip() == ""
    r0 = subprocess.run(cmd, env=dict(env, RANK="0", LOCAL_RANK="0"), capture_output=True, text=True, timeout=300)
    assert r0.returncode == 0, r0.stderr
    line = json.loads(r0.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["n_gpus"] == 2 and line["value"] > 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["e2e"]["h2d_bytes_per_step"] == 0
