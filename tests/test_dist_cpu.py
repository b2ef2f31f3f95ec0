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


def test_bench_accounting_matches_the_survey_tables():
    """bench.py's algorithmic work: causal pairs, two-pass flops and minimum bytes of
    configs 2-4, and the committed ncu summaries the `roofline.traffic` key is read from at run time."""
    import bench
    from paper_2606_07577_b200 import inputs as I
    want = {2: (107.35e6, 43.09e12, 6.12e9), 3: (429.38e6, 253.26e12, 26.47e9), 4: (31.59e6, 18.63e12, 6.16e9)}
    for cfg, (pairs, flops, nbytes) in want.items():
        wl = I.CONFIGS[cfg]
        w = bench.algorithmic_work(wl, wl.n_v, wl.n_a)
        assert abs(w["pairs"] - pairs) < 0.01e6 * 1.5 and abs(2 * w["f_pass"] - flops) < 0.01e12 and abs(w["bytes"]["total"] - nbytes) < 0.01e9
        assert w["exps_pass"] == w["pairs"] * wl.Hq * wl.L and w["Nk"] == wl.n_v + wl.n_a + wl.Nn
    # DRAM traffic per launch of the two scoring passes, read from profiles/: within 5 % of the algorithmic Q + K bytes
    for name, cfg in (("cfg2_qwen25omni7b", 2), ("cfg3_8b", 3), ("cfg4_4b_tight", 4)):
        wl = I.CONFIGS[cfg]
        qk = (wl.L * wl.Hq * wl.Nn + wl.L * wl.Hkv * (wl.n_v + wl.n_a + wl.Nn)) * wl.D * 2
        for pass_no in (1, 2):
            traffic, src = bench.ncu_traffic(name, f"score_tc_kernel<{pass_no}")
            assert traffic is not None and src.startswith("profiles/"), src
            assert 1.0 <= traffic / qk < 1.05, (name, pass_no, traffic / qk)
    assert bench.ncu_traffic("cfg1_tiny_fp32", "score_tc_kernel<1")[0] is None     # no capture committed: null, with the reason as source
