"""The N > 1 path of bench.py on CPU: world_size 2, gloo backend.  north_star fixes one GPU and no data-path
collective, so ranks are independent replicas; what N > 1 adds is the max-over-ranks timing and
the whole-job aggregate, and the reference arm running on rank 0 only."""
import os
import pathlib
import subprocess
import sys

import torch.multiprocessing as mp

ROOT = pathlib.Path(__file__).resolve().parents[1]


def _worker(rank, world, port, out):
    import torch.distributed as dist

    sys.path.insert(0, str(ROOT))
    import bench

    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ms_local = 10.0 + 5.0 * rank                      # rank 1 is the slow replica
    ms, value = bench.whole_job(ms_local, units_per_rank=30, world=world, device="cpu")
    dist.barrier()
    dist.destroy_process_group()
    out.put((rank, ms, value))


def test_whole_job_is_max_over_ranks_and_sums_replicas():
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    got = sorted(out.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, ms, value in got:
        assert ms == 15.0                              # the slowest replica
        assert abs(value - 2 * 30 / 15e-3) < 1e-9      # units of BOTH replicas over that time


def test_single_rank_needs_no_process_group():
    sys.path.insert(0, str(ROOT))
    import bench

    assert bench.whole_job(4.0, 12, 1, "cpu") == (4.0, 3000.0)


def test_reference_arm_runs_on_rank_0_only():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    r = subprocess.run([sys.executable, str(ROOT / "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1",
                        "--warmup", "0"], env=env, capture_output=True, text=True, timeout=300)
    assert r.returncode == 0 and r.stdout.strip() == ""
