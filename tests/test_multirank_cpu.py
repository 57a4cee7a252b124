"""N > 1 bookkeeping of bench.py on the CPU (gloo, world_size 2): frames are independent, so ranks share no
data-path collective; the only exchange is the max-over-ranks of the timed region."""
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    import torch
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    sys.path.insert(0, os.path.join(ROOT, "tests"))
    import bench
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)

    def all_max(x):
        t = torch.tensor([x], dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        return float(t[0])

    ms_local = 10.0 * (rank + 1)                    # rank 1 is the slow one
    fps, ms = bench.whole_job(300, world, ms_local, all_max)
    assert bench.dist_env() == (rank, 0, world) or bench.dist_env()[0] == rank
    out.put((rank, fps, ms))
    dist.barrier()
    dist.destroy_process_group()


def test_whole_job_value_is_all_frames_over_the_slowest_rank():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(2))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, fps, ms in res:
        assert ms == pytest.approx(20.0)
        assert fps == pytest.approx(2 * 300 / 20e-3)


def test_single_process_value():
    sys.path.insert(0, ROOT)
    import bench
    fps, ms = bench.whole_job(300, 1, 12.5)
    assert ms == 12.5 and fps == pytest.approx(300 / 12.5e-3)


def test_reference_arm_other_ranks_exit_without_work():
    env = dict(os.environ, RANK="1", LOCAL_RANK="1", WORLD_SIZE="2")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", "1",
                        "--warmup", "0", "--gpus", "2"], env=env, capture_output=True, text=True, timeout=120)
    assert r.returncode == 0 and r.stdout.strip() == ""


def test_gpus_flag_without_a_launcher_starts_the_ranks_itself():
    """`python bench.py --gpus 2` with WORLD_SIZE unset goes through bench.launch_ranks (torch.distributed.run,
    2 ranks) and prints ONE line with n_gpus = 2; the CPU stand-in uses gloo and a sleep for the kernels."""
    import json
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "LOCAL_RANK", "WORLD_SIZE", "MASTER_ADDR", "MASTER_PORT")}
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--selftest-launch"], env=env,
                       capture_output=True, text=True, timeout=300)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [ln for ln in r.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1, r.stdout
    rec = json.loads(lines[0])
    assert rec["n_gpus"] == 2 and rec["ms_per_step"] == pytest.approx(20.0)
    assert rec["value"] == pytest.approx(2 * 300 / 20e-3)


def test_gpus_flag_fails_loudly_when_the_devices_are_missing():
    """No silent 1-GPU run: asking for more GPUs than are visible exits non-zero and prints no JSON line."""
    import torch
    if torch.cuda.device_count() >= 2:
        pytest.skip("two CUDA devices are present")
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "LOCAL_RANK", "WORLD_SIZE")}
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--steps", "1"], env=env,
                       capture_output=True, text=True, timeout=300)
    assert r.returncode != 0 and "{" not in r.stdout
