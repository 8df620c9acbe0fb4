"""Host-side logic of bench.py that the N > 1 launch relies on, exercised with world_size 2 over gloo on CPU
(the path does not shard -- DESIGN.md section 8, "replicas only" -- so the only cross-rank step is the
max-over-ranks of the timing and the aggregation of the replicas' throughput)."""
import json
import os
import subprocess
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    t = bench.max_over_ranks(10.0 + 5.0 * rank)                  # rank 1 is the slow one
    v = bench.aggregate_value(1000, 4, t, world)
    dist.barrier()
    with open(f"{out}.{rank}", "w") as f:
        json.dump({"t": t, "v": v}, f)
    dist.destroy_process_group()


def test_timing_is_max_over_ranks_and_value_is_whole_job(tmp_path):
    world, out = 2, str(tmp_path / "r")
    mp.spawn(_worker, args=(world, 29671, out), nprocs=world, join=True)
    res = [json.load(open(f"{out}.{r}")) for r in range(world)]
    for r in res:
        assert r["t"] == 15.0                                    # the max, on every rank
        assert r["v"] == 2 * 1000 * 4 / 15.0e-3                  # both replicas' cells over the slowest rank's time


def test_single_process_needs_no_process_group():
    import bench
    assert bench.max_over_ranks(3.5) == 3.5
    assert bench.aggregate_value(10, 2, 4.0, 1) == 10 * 2 / 4.0e-3


def test_reference_arm_runs_on_rank_0_only():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2"],
                       env=env, capture_output=True, text=True, timeout=120)
    assert r.returncode == 0 and r.stdout.strip() == ""


def test_counters_are_tied_to_the_kernel_sources(tmp_path, monkeypatch):
    """bench.py prints ncu-derived numbers only while the hash stored with them equals the hash of csrc/ (VERDICT r1 item 9)."""
    from paper_2409_16053_b200 import counters
    sha = counters.csrc_sha()
    assert len(sha) == 16 and sha == counters.csrc_sha()
    prof = tmp_path / "profiles"
    prof.mkdir()
    monkeypatch.setattr(counters, "ROOT", str(tmp_path))
    assert counters.load("cfg3") is None                                   # no file
    (prof / "r02_stage_counters_cfg3.json").write_text(json.dumps({"csrc_sha": "0" * 16, "launches": {}}))
    assert counters.load("cfg3") is None                                   # stale: taken on other sources
    (prof / "r02_stage_counters_cfg3.json").write_text(json.dumps({"csrc_sha": sha, "launches": {"stage1": {}}}))
    assert counters.load("cfg3")["launches"] == {"stage1": {}}
    # a raw-page CSV as ncu writes it: header row, units row, one row per launch
    csv_path = tmp_path / "c.csv"
    hdr = ["ID", "Kernel Name", "gpu__time_duration.sum", "dram__bytes_read.sum", "dram__bytes_write.sum", "sm__inst_executed_pipe_fp64.sum"]
    rows = [hdr, ["", "", "ns", "byte", "byte", "inst"],
            ["0", "void ak::stage_v3_kernel<1, 0, 16, 10, 2, 0>(CUtensorMap_st)", "10,000", "4", "2", "100"],
            ["1", "void ak::stage_v3_kernel<1, 0, 16, 10, 2, 1>(CUtensorMap_st)", "12,000", "8", "2", "110"],
            ["2", "void ak::stage_v3_kernel<1, 0, 16, 10, 2, 0>(CUtensorMap_st)", "20,000", "6", "2", "100"]]
    csv_path.write_text("\n".join(",".join(f'"{c}"' for c in r) for r in rows))
    d = counters.parse(str(csv_path), "cfg3")
    assert d["launches"]["stage1"]["gpu__time_duration.sum"] == 15000.0 and d["launches"]["stage1"]["launches_averaged"] == 2
    assert d["launches"]["stage2"]["dram__bytes_read.sum"] == 8.0 and d["csrc_sha"] == sha
