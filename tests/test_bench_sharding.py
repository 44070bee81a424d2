"""CPU tests (world_size 2, gloo) of the N > 1 host logic of bench.py: the path shards by candidate
with no data-path collective ("replicas only"); the only cross-rank datum is the
max-over-ranks time, and the reference arm runs on rank 0 alone."""
import json
import os
import subprocess
import sys
from pathlib import Path

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = Path(__file__).resolve().parents[1]
sys.path.insert(0, str(ROOT))
import bench  # noqa: E402


def _worker(rank, world, port, out_dir):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    mine = [1.0 + rank, 5.0 - rank, 2.0]                       # per-rank "timings"
    red = bench.reduce_max(mine, device="cpu")
    seed = bench.rank_x0_seed(1, rank)
    dist.barrier()
    Path(out_dir, f"r{rank}.json").write_text(json.dumps({"red": red, "seed": seed}))
    dist.destroy_process_group()


def test_max_over_ranks_and_distinct_batches(tmp_path):
    world, port = 2, 29500 + os.getpid() % 2000
    mp.spawn(_worker, args=(world, port, str(tmp_path)), nprocs=world, join=True)
    r = [json.loads(Path(tmp_path, f"r{i}.json").read_text()) for i in range(world)]
    assert r[0]["red"] == r[1]["red"] == [2.0, 5.0, 2.0]       # element-wise max over the two ranks
    assert r[0]["seed"] != r[1]["seed"]                         # every replica draws its own candidates
    # whole-job value: all ranks' evaluations over the slowest rank's time
    assert bench.whole_job_value(2, 10, 4, 3, 2.0) == 2 * 10 * 4 * 3 / 2.0


def test_reduce_max_single_process():
    assert bench.reduce_max([3.0, 1.0]) == [3.0, 1.0]


def test_reference_arm_runs_on_rank0_only():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    p = subprocess.run([sys.executable, str(ROOT / "bench.py"), "--impl", "reference", "--gpus", "2", "--config", "0",
                        "--steps", "1", "--warmup", "0"], env=env, capture_output=True, text=True, timeout=300)
    assert p.returncode == 0 and p.stdout.strip() == ""
    env["RANK"] = "0"
    p = subprocess.run([sys.executable, str(ROOT / "bench.py"), "--impl", "reference", "--gpus", "2", "--config", "0",
                        "--steps", "1", "--warmup", "0"], env=env, capture_output=True, text=True, timeout=300)
    line = json.loads(p.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["cpu_baseline"]["kind"] == "oracle" and line["value"] > 0
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["n_gpus"] == 2
