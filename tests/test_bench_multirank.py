"""Host logic of bench.py's N > 1 path ("replicas only") on CPU: two gloo
ranks reduce their step times to the slowest one and rank 0 forms the whole-job throughput."""
import os
import socket
import sys

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, times, out_path):
    sys.path.insert(0, ROOT)
    import bench
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    dist.barrier()
    ms = bench.max_over_ranks(times[rank], dist, device="cpu")
    if rank == 0:
        with open(out_path, "w") as f:
            f.write(f"{ms!r} {bench.whole_job_gflops(world, 1000, ms)!r}")
    dist.destroy_process_group()


def test_two_ranks_take_the_slowest_time(tmp_path):
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    out = tmp_path / "r0.txt"
    times = [1.25, 2.5]
    mp.spawn(_worker, args=(2, port, times, str(out)), nprocs=2, join=True)
    ms, gf = (float(x) for x in out.read_text().split())
    assert ms == 2.5
    # 2 ranks x 2 half-Dhops x 1320 flop x 1000 sites in 2.5 ms
    assert gf == pytest.approx(2 * 2 * 1320 * 1000 / 2.5e-3 / 1e9)


def test_single_rank_is_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks(3.0) == 3.0
    assert bench.whole_job_gflops(1, 8388608, 1.0) == pytest.approx(2 * 1320 * 8388608 / 1e-3 / 1e9)


def test_gpus_flag_starts_that_many_ranks(tmp_path):
    """`python bench.py --gpus 2` without a launcher starts two ranks under torch.distributed.run (127.0.0.1): on this
    CPU box each rank gets as far as the first CUDA call and stops there with its rank and the world size in the message."""
    import subprocess
    code = ("import sys; sys.path.insert(0, %r); import bench; "
            "sys.exit(bench.spawn_ranks(2, ['--gpus', '2', '--steps', '1', '--warmup', '3', '--no-cpu'], check_devices=False))" % ROOT)
    env = dict(os.environ, CUDA_VISIBLE_DEVICES="")
    env.pop("WORLD_SIZE", None)
    r = subprocess.run([sys.executable, "-c", code], capture_output=True, text=True, env=env, timeout=600)
    assert r.returncode != 0
    out = r.stdout + r.stderr
    assert "no CUDA device for rank 0 of 2" in out and "no CUDA device for rank 1 of 2" in out, out[-2000:]
