"""Host-side logic of bench.py: work model constants, the multi-rank (N > 1) timing reduction over gloo with
world_size 2, and the --impl reference arm (the oracle timed on host cores; no GPU needed)."""
import json
import os
import subprocess
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_work_model_matches_survey_table():
    import bench
    assert [int(bench.flops_eval(n)) for n in (128, 256, 512, 1024)] == [103040, 208640, 422400, 855040]
    assert int(bench.bytes_eval(256)) == 12360
    assert abs(bench.FP64_PEAK_TFLOPS - 37.2) < 0.05


def _worker(rank, world, port, q):
    import torch.distributed as dist
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    sys.path.insert(0, ROOT)
    import bench
    ids = bench.shard_info(rank, world, 360)
    t = bench.max_over_ranks(10.0 + 5.0 * rank, dist)
    q.put((rank, int(ids[0]), int(ids[-1]), len(ids), t))
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_sharding_and_max_time_gloo():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + (os.getpid() % 2000)
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(2))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert res[0][:4] == (0, 0, 359, 360) and res[1][:4] == (1, 360, 719, 360)     # disjoint replicas
    assert res[0][4] == 15.0 and res[1][4] == 15.0                                  # max over ranks on both


def test_reference_arm_prints_contract_line():
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", "1",
                          "--warmup", "3"], capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert out.returncode == 0, out.stderr[-2000:]
    line = json.loads(out.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["unit"] == "evals/s" and line["value"] > 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["cpu_baseline"]["cores"] >= 1
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["gpu_launches"] == 0
    assert line["config"]["workload"].startswith("cfg5")


def test_reference_arm_nonzero_rank_exits_quietly():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2")
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2"],
                         capture_output=True, text=True, timeout=120, cwd=ROOT, env=env)
    assert out.returncode == 0 and out.stdout.strip() == ""
