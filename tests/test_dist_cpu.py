"""Multi-process host logic of bench.py on CPU (gloo, world_size 2): the path does not shard (DESIGN.md section 9,
"replicas only"), so the only cross-rank step is the MAX-reduce of the timing scalars and the whole-job value."""
import json
import os
import socket
import subprocess
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, world: int, port: int, out_dir: str):
    import bench
    os.environ["MASTER_ADDR"], os.environ["MASTER_PORT"] = "127.0.0.1", str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        mine = [10.0 + rank, 3.0 - rank, 0.5]                      # rank 0: 10, 3, .5   rank 1: 11, 2, .5
        got = bench.max_over_ranks(mine, torch.device("cpu"), world)
        value = bench.job_value(world, 21980, got[0] / 4)          # 4 steps
        with open(os.path.join(out_dir, f"r{rank}.json"), "w") as f:
            json.dump({"got": got, "value": value}, f)
    finally:
        dist.destroy_process_group()


def test_max_over_ranks_and_job_value_gloo(tmp_path):
    world = 2
    mp.spawn(_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    res = [json.load(open(tmp_path / f"r{r}.json")) for r in range(world)]
    for r in res:                                                   # every rank sees the slowest rank's times
        assert r["got"] == [11.0, 3.0, 0.5]
        assert abs(r["value"] - 2 * 21980 / (11.0 / 4)) < 1e-9      # both replicas' units over the max time


def test_single_rank_is_identity():
    import bench
    assert bench.max_over_ranks([1.5, 2], torch.device("cpu"), 1) == [1.5, 2.0]
    assert bench.job_value(1, 100, 0.5) == 200.0


def test_reference_arm_only_rank0_works():
    """`bench.py --impl reference` under a 2-rank launch: rank 1 exits 0 without work and prints nothing."""
    env = dict(os.environ, RANK="1", LOCAL_RANK="1", WORLD_SIZE="2", MASTER_ADDR="127.0.0.1", MASTER_PORT=str(_free_port()))
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--config", "1",
                        "--steps", "1", "--warmup", "0"], env=env, capture_output=True, text=True, timeout=300)
    assert r.returncode == 0 and r.stdout.strip() == ""
    env["RANK"], env["LOCAL_RANK"] = "0", "0"
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--config", "1",
                        "--steps", "1", "--warmup", "0"], env=env, capture_output=True, text=True, timeout=300)
    assert r.returncode == 0
    line = json.loads(r.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["cpu_baseline"]["kind"] == "oracle" and line["value"] > 0
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["n_gpus"] == 2
