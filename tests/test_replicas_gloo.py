"""N > 1 path of bench.py on CPU: replicas only.  Two gloo ranks each "advance" their own copy of a
workload in a different time; the aggregate must use the MAX over ranks and count both ranks' cell updates, and the
reference arm must print on rank 0 only."""
import json
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


def _worker(rank, world, port, q):
    import torch.distributed as dist

    sys.path.insert(0, ROOT)
    import bench

    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ms_local = 10.0 if rank == 0 else 25.0  # rank 1 is the slow replica
    ms, value = bench.replicas_aggregate(ms_local, cells=1000, steps=5, world=world)
    dist.barrier()
    dist.destroy_process_group()
    q.put((rank, ms, value))


def test_replicas_aggregate_world2():
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
    for rank, ms, value in got:
        assert ms == 25.0  # max over ranks, on every rank
        assert abs(value - 1000 * 5 * 2 / 25e-3 / 1e9) < 1e-12  # both replicas' cell updates over the slowest time


def test_replicas_aggregate_single():
    sys.path.insert(0, ROOT)
    import bench

    ms, value = bench.replicas_aggregate(4.0, cells=2 ** 20, steps=3, world=1)
    assert ms == 4.0 and abs(value - 2 ** 20 * 3 / 4e-3 / 1e9) < 1e-12


def test_reference_arm_prints_on_rank0_only():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1",
                          "--warmup", "0", "--config", "1"], env=env, capture_output=True, text=True, timeout=300)
    assert out.returncode == 0 and out.stdout.strip() == ""
    env["RANK"] = "0"
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1",
                          "--warmup", "0", "--config", "1"], env=env, capture_output=True, text=True, timeout=300)
    assert out.returncode == 0, out.stderr
    line = json.loads(out.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["value"] > 0 and line["cpu_baseline"]["kind"] == "oracle"
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["e2e"]["d2h_bytes_per_step"] == 0
