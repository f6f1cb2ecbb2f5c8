"""Host logic of bench.py's N > 1 path on CPU (gloo, world_size 2).

The path does not shard (replicas only): every rank runs its own copy of the
workload, there is no data-path collective, and the only communication is the barrier and the
MAX over ranks of the device time.  These tests run that aggregation through a real process group
and check the reference arm's rank-0-only contract."""
import json
import os
import socket
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, q):
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    import bench
    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    local_seconds = 2.0 + 0.5 * rank            # rank 1 is the slow replica
    dist.barrier()
    mx = bench.max_over_ranks(local_seconds, world)
    val = bench.whole_job_value(cells_per_replica=1000, steps=4, world=world, seconds_max=mx)
    q.put((rank, mx, val))
    dist.barrier()
    dist.destroy_process_group()


def test_replica_aggregation_gloo_world2():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    out = sorted(q.get(timeout=120) for _ in range(2))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, mx, val in out:
        assert mx == 2.5                         # max over ranks, identical on every rank
        assert val == 2 * 1000 * 4 / 2.5         # whole-job aggregate over both replicas
    assert [r for r, _, _ in out] == [0, 1]


def test_single_rank_aggregation_is_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks(3.25, 1) == 3.25
    assert bench.whole_job_value(10, 2, 1, 4.0) == 5.0


@pytest.mark.slow
def test_reference_arm_rank1_is_silent_and_rank0_prints_one_json_line():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                        "--steps", "1", "--warmup", "0"], env=env, capture_output=True, text=True, timeout=120)
    assert r.returncode == 0 and r.stdout.strip() == ""
    env = dict(os.environ, RANK="0", WORLD_SIZE="2", LOCAL_RANK="0")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                        "--steps", "1", "--warmup", "0", "--oracle-crop", "96"], env=env, capture_output=True,
                       text=True, timeout=300)
    assert r.returncode == 0, r.stderr
    lines = [l for l in r.stdout.splitlines() if l.strip()]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["value"] > 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["e2e"]["h2d_bytes_per_step"] == 0
    assert d["config"]["oracle_crop"] == 96 and "96x96" in d["cpu_baseline"]["sample"]
    assert d["unit"] == "cell-updates/s" and d["higher_is_better"] is True
