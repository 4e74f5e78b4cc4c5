"""The N > 1 path of bench.py on CPU: two gloo ranks, "replicas only" aggregation (MAX over ranks of
the elapsed time, whole-job value = N * steps / max time), and the reference arm's rank-0-only rule."""
import json
import os
import subprocess
import sys

import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    import bench
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ms = 100.0 if rank == 0 else 125.0          # rank 1 is the slow one
    agg = bench.aggregate_over_ranks(ms, ms / 10 * 1.5, steps=10, world=world)
    json.dump(agg, open(f"{out}.{rank}", "w"))
    dist.barrier()
    dist.destroy_process_group()


def test_replicas_aggregation_gloo_world2(tmp_path):
    out = str(tmp_path / "agg")
    mp.spawn(_worker, args=(2, 29613, out), nprocs=2, join=True)
    a, b = (json.load(open(f"{out}.{r}")) for r in (0, 1))
    assert a == b
    assert a["ms_total"] == 125.0 and abs(a["ms_per_step"] - 12.5) < 1e-12
    assert abs(a["value"] - 2 * 10 / 0.125) < 1e-9          # whole-job iterations/s over both replicas
    assert abs(a["e2e_value"] - 2 * 1e3 / 18.75) < 1e-9


def test_single_rank_aggregation_is_identity():
    sys.path.insert(0, ROOT)
    import bench
    a = bench.aggregate_over_ranks(50.0, 6.0, steps=5, world=1)
    assert a["ms_per_step"] == 10.0 and a["value"] == 100.0 and abs(a["e2e_value"] - 1e3 / 6.0) < 1e-12


def test_reference_arm_only_rank0_prints():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "cfg0",
                        "--steps", "2", "--warmup", "1"], env=env, capture_output=True, text=True, timeout=120)
    assert r.returncode == 0 and r.stdout.strip() == ""
    env = dict(os.environ, RANK="0", WORLD_SIZE="2", LOCAL_RANK="0")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "cfg0",
                        "--steps", "2", "--warmup", "1", "--gpus", "2"], env=env, capture_output=True, text=True,
                       timeout=120)
    line = json.loads(r.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["unit"] == "iterations/s" and line["value"] > 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["e2e"]["h2d_bytes_per_step"] == 0
