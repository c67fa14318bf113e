"""Host-side logic of bench.py's N > 1 path on CPU: world-size-2 gloo, MAX-over-ranks timing and
whole-job throughput ("replicas only": ranks exchange one scalar, never field data), and the
reference arm's rank handling."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, q):
    import torch
    import torch.distributed as td
    sys.path.insert(0, ROOT)
    import bench
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    td.init_process_group("gloo", rank=rank, world_size=world)
    dev = torch.device("cpu")
    ms_local = 10.0 + 5.0 * rank            # rank 1 is the slow one
    glups, ms = bench.job_glups(1000_000, 7, ms_local, world, dev)
    mx = bench.max_over_ranks(float(rank), world, dev)
    td.barrier()
    td.destroy_process_group()
    q.put((rank, glups, ms, mx))


def test_two_rank_gloo_aggregation():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, glups, ms, mx in res:
        assert ms == 15.0                       # the max over ranks, on every rank
        assert mx == 1.0
        assert glups == pytest.approx(2 * 1000_000 * 7 / 15e-3 / 1e9)


def test_single_rank_is_identity():
    sys.path.insert(0, ROOT)
    import bench
    g, ms = bench.job_glups(10, 2, 4.0, 1, None)
    assert ms == 4.0 and g == pytest.approx(10 * 2 / 4e-3 / 1e9)


def test_reference_arm_runs_on_rank0_only():
    """`bench.py --impl reference`: rank 0 prints one JSON line with impl=reference, e2e and
    cpu_baseline; any other rank exits 0 without work."""
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference",
                        "--steps", "2", "--warmup", "1", "--n", "256"], env=env,
                       capture_output=True, text=True, timeout=300)
    assert r.returncode == 0 and r.stdout.strip() == ""
    env = dict(os.environ, RANK="0", WORLD_SIZE="1", LOCAL_RANK="0")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference",
                        "--steps", "2", "--warmup", "1", "--n", "256"], env=env,
                       capture_output=True, text=True, timeout=300)
    assert r.returncode == 0
    lines = [l for l in r.stdout.splitlines() if l.strip()]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["cpu_baseline"]["kind"] == "oracle"
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["value"] > 0
    assert d["steps"] == 2
