"""Host-side logic of bench.py that has no GPU in it: the N > 1 aggregation (max-over-ranks time, summed units) over a
world_size-2 gloo group, the reference arm's rank gating, and the JSON contract of `--impl reference`."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, q):
    # the environment torchrun gives every rank; the group is created by bench.py's own init_dist (the code path of
    # `bench.py --gpus N`: NCCL + gloo with GPUs, gloo alone here) and the host barrier / aggregation are bench.py's
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world), LOCAL_RANK=str(rank))
    sys.path.insert(0, ROOT)
    import bench
    assert bench.dist_env() == (rank, world, rank)
    dist = bench.init_dist(world)
    bench.host_barrier(dist)
    ms, units = bench.aggregate(10.0 + 5.0 * rank, 100.0 * (rank + 1), world, dist)
    # every rank draws its own Monte-Carlo samples
    a = bench.make_input("c1", 16, 1, rank)
    q.put((rank, ms, units, float(a.sum())))
    bench.host_barrier(dist)
    dist.destroy_process_group()


def test_aggregate_world_size_2_gloo():
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
    for _, ms, units, _chk in res:
        assert ms == 15.0          # max over ranks
        assert units == 300.0      # whole-job units
    assert res[0][3] != res[1][3]  # seeds offset by rank


def test_aggregate_single_rank_is_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.aggregate(3.5, 7.0, 1, None) == (3.5, 7.0)


def test_reference_arm_contract():
    env = dict(os.environ, OMP_NUM_THREADS="4")
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--workload", "c1", "--steps", "1",
                          "--warmup", "0"], capture_output=True, text=True, env=env, timeout=600)
    assert out.returncode == 0, out.stderr
    line = json.loads(out.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["unit"] == "grid-point-stages/s" and line["higher_is_better"] is True
    assert line["value"] > 0 and line["cpu_baseline"]["kind"] == "oracle" and line["cpu_baseline"]["cores"] >= 1
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["e2e"]["d2h_bytes_per_step"] == 0
    # ranks other than 0 exit 0 without work
    env["RANK"], env["WORLD_SIZE"] = "1", "2"
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--workload", "c1"],
                         capture_output=True, text=True, env=env, timeout=120)
    assert out.returncode == 0 and out.stdout.strip() == ""
