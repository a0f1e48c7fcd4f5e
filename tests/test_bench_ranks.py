"""The N > 1 path of bench.py on CPU: two gloo ranks (replicas only) - timing is the max over
ranks, the value is the whole-job aggregate, and the reference arm runs on rank 0 only."""
import os
import socket
import subprocess
import sys
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parents[1]


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    import torch
    import torch.distributed as dist
    sys.path.insert(0, str(ROOT))
    import bench
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    total_ms, e2e_ms = bench.max_over_ranks([100.0 + 50.0 * rank, 7.0 - rank], dist, torch.device("cpu"))
    dist.barrier()
    dist.destroy_process_group()
    out.put((rank, total_ms, e2e_ms, bench.whole_job_value(world, 1000.0, total_ms)))


def test_two_rank_aggregation_gloo():
    import torch.multiprocessing as mp
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
    for rank, total_ms, e2e_ms, value in res:
        assert total_ms == 150.0 and e2e_ms == 7.0            # max over ranks, identical on every rank
        assert value == pytest.approx(2 * 1000.0 / 0.150)     # whole-job aggregate of 2 replicas


def test_reference_arm_other_ranks_do_no_work():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2")
    r = subprocess.run([sys.executable, str(ROOT / "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1",
                        "--warmup", "0"], env=env, capture_output=True, text=True, timeout=120)
    assert r.returncode == 0 and r.stdout.strip() == ""


def test_gpus_n_starts_n_ranks_itself():
    """`python bench.py --gpus N` without a launcher re-executes itself under torch.distributed.run with N processes (so the line
    it prints says n_gpus = N); under a launcher (WORLD_SIZE set) and for one GPU it starts nothing."""
    sys.path.insert(0, str(ROOT))
    import bench
    argv = ["--gpus", "4", "--steps", "2", "--warmup", "3", "--shard"]
    cmd = bench.self_launch_command(4, argv, {})
    assert cmd[:3] == [sys.executable, "-m", "torch.distributed.run"]
    assert "--nproc-per-node=4" in cmd and "--nnodes=1" in cmd
    assert cmd[cmd.index("--master-addr") + 1] == "127.0.0.1" and int(cmd[cmd.index("--master-port") + 1]) > 0
    assert cmd[-len(argv) - 1:] == [str(ROOT / "bench.py"), *argv]
    assert bench.self_launch_command(4, argv, {"WORLD_SIZE": "4"}) is None
    assert bench.self_launch_command(1, ["--gpus", "1"], {}) is None


def test_gpus_n_on_a_box_without_gpus_fails_loudly():
    """The self-started ranks find no device: non-zero exit and a message, never a CPU result."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    r = subprocess.run([sys.executable, str(ROOT / "bench.py"), "--gpus", "2", "--steps", "1", "--warmup", "0", "--config", "0"],
                       capture_output=True, text=True, timeout=300)
    assert r.returncode != 0 and "no CPU fallback" in (r.stderr + r.stdout)
    assert "point-updates/s" not in r.stdout
