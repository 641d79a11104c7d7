"""CPU coverage of bench.py's N>1 host logic (replicas only): world-size-2 gloo
rendezvous on 127.0.0.1, max-over-ranks timing, whole-job aggregation; --impl reference rank gating."""
import json
import os
import subprocess
import sys

import pytest
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out_dir):
    os.environ.update(RANK=str(rank), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    sys.path.insert(0, ROOT)
    import bench
    dist = bench.init_dist(world, rank, backend="gloo")
    local_ms = 10.0 + 5.0 * rank                      # rank 1 is the slow one
    ms = bench.max_over_ranks(local_ms, dist, "cpu")
    dist.barrier()
    val = bench.whole_job_value(world, 1_000_000_000, ms)
    json.dump({"ms": ms, "value": val}, open(os.path.join(out_dir, f"r{rank}.json"), "w"))
    dist.destroy_process_group()


def test_two_rank_gloo_max_and_aggregate(tmp_path):
    world = 2
    mp.spawn(_worker, args=(world, 29533, str(tmp_path)), nprocs=world, join=True)
    res = [json.load(open(tmp_path / f"r{r}.json")) for r in range(world)]
    for r in res:
        assert r["ms"] == 15.0                        # max over ranks, identical on every rank
        assert abs(r["value"] - 2 * 1e9 / 15e-3 / 1e9) < 1e-9   # 2 replicas' bytes / slowest time


def test_single_rank_helpers_need_no_process_group():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.init_dist(1, 0) is None
    assert bench.max_over_ranks(3.5, None) == 3.5
    assert bench.whole_job_value(1, 2_000_000_000, 1.0) == 2000.0


def test_reference_arm_nonzero_rank_exits_quietly():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    p = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                        "--steps", "1", "--warmup", "0"], env=env, capture_output=True, text=True, timeout=300)
    assert p.returncode == 0 and p.stdout.strip() == ""


def test_ncu_traffic_reads_a_raw_page_and_rewrites_one_row(tmp_path, golden_dir):
    """paper_2510_20171_b200.ncu_traffic: the committed tool behind bench.py's `roofline.traffic` (tests/golden/
    ncu_raw_page_sample.csv = the round-3 capture's raw page trimmed to the columns it reads)."""
    import csv
    import os
    from paper_2510_20171_b200 import ncu_traffic as T
    rd, wr = T.dram_bytes(os.path.join(golden_dir, "ncu_raw_page_sample.csv"), "segment_copy_kernel")
    assert (rd, wr) == (10737655000, 10683552000)
    assert abs((rd + wr) / (2 * 10 * 2**30) - 1) < 0.01          # within 1 % of config 3's algorithmic bytes
    p = tmp_path / "traffic.csv"
    T.update(str(p), "k", "w", 1, 2, "first")
    T.update(str(p), "k2", "w", 5, 6, "other")
    T.update(str(p), "k", "w", 3, 4, "second")                   # replaces the first row
    rows = list(csv.DictReader(open(p)))
    assert [(r["kernel"], r["bytes_per_launch"], r["source"]) for r in rows] == [("k2", "11", "other"), ("k", "7", "second")]
