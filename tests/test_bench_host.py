"""CPU-only checks of bench.py's host logic: the byte model, the reference arm's JSON line and
the N>1 reduction (world_size-2 gloo group; the data path itself has no collective -- replicas
only)."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_algorithmic_bytes_match_survey_table():
    import bench
    cfg = dict(n=10_000_000, nq=10_000_000, dim=3, pkind=0, qkind=2, k=16)
    b = bench.algorithmic_bytes(cfg, dict(pairs=159_000_000))
    n = cfg["n"]
    assert b["B1_bounds"] == 12 * n                                   # 12 B/prim
    assert b["B2_codes"] == 20 * n
    assert bench.sort_passes(n, 3) == 5                               # 13 bits per axis at N = 10^7
    assert b["B3_sort_hist"] + b["B3_sort_pass"] == (8 + 20 + 4 * 24) * n
    assert b["B4_leaves"] == 32 * n
    assert b["B5B6_hierarchy_refit"] == 92 * n                        # B5 20 + B6 72
    assert b["T2_scan"] == 12 * n + 4
    # traversal: per query 4 (order) + 16 (query) + 4 (count); tree = 48 B per TOUCHED primitive
    t = bench.algorithmic_bytes(cfg, dict(pairs=159_000_000, touched_spatial=460_000, touched_knn=460_000))
    assert t["T1_spatial_count"] == 2 * (24 * n + 48 * 460_000) + 4 * 159_000_000
    assert t["K1K2_knn"] == n * (4 + 12 + 8 * 16) + 48 * 460_000     # = 1.46 GB at C3
    assert b["_whole_tree"] == 4 * (n * 4 + (n - 1) * 16)
    # boxes (C4) and 5-D points (C5): SURVEY.md's 88 + 20 and 112 + 20 bytes per primitive
    assert bench.algorithmic_bytes(dict(n=100, nq=10, dim=3, pkind=1, qkind=1, k=None), dict(pairs=0))["B5B6_hierarchy_refit"] == 108 * 100
    assert bench.algorithmic_bytes(dict(n=100, nq=10, dim=5, pkind=0, qkind=2, k=8), dict(pairs=0))["B5B6_hierarchy_refit"] == 132 * 100


def test_reference_arm_prints_contract_line():
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--workload", "C1",
                          "--steps", "1", "--warmup", "0"], capture_output=True, text=True, check=True, cwd=ROOT)
    line = json.loads(out.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["unit"] == "queries/s" and line["value"] > 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["cpu_baseline"]["cores"] >= 1
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["e2e"]["value"] == line["value"]
    assert line["config"] == dict(workload="C1", n=10000, nq=10000, dim=3, k=10, r=0.062)
    assert line["extrapolated_from_queries"] is None and "measured" in line["full_step_source"]


_WORKER = r"""
import os, sys
sys.path.insert(0, {root!r})
import torch.distributed as dist
import bench
dist.init_process_group("gloo", init_method="tcp://127.0.0.1:{port}", rank=int(sys.argv[1]), world_size=2)
r = dist.get_rank()
got = bench.max_over_ranks([10.0 + r, 5.0 - r])
assert got == [11.0, 5.0], got
assert bench.rank_seed_offset(r) == 1000 * r
from paper_2507_23700_b200 import datagen as dg
a = dg.config("C1", 0.01, seed_offset=bench.rank_seed_offset(r))["prims"]
import torch
t = torch.tensor([float(a.sum())], dtype=torch.float64)
both = [torch.zeros_like(t) for _ in range(2)]
dist.all_gather(both, t)
assert float(both[0]) != float(both[1])      # replicas draw distinct inputs
dist.destroy_process_group()
print("ok", r)
"""


def test_max_over_ranks_gloo_world2(tmp_path):
    port = 29000 + os.getpid() % 2000
    script = tmp_path / "w.py"
    script.write_text(_WORKER.format(root=ROOT, port=port))
    procs = [subprocess.Popen([sys.executable, str(script), str(r)], stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True)
             for r in range(2)]
    for p in procs:
        out, err = p.communicate(timeout=120)
        assert p.returncode == 0, err
        assert out.startswith("ok")


def test_gpus_flag_starts_the_ranks_itself():
    """`python bench.py --gpus 2` outside torchrun re-executes itself under torch.distributed.run
    with 2 ranks (it used to run one rank and print n_gpus 1).  Checked on the
    reference arm, which needs no GPU: rank 0 prints the line, rank 1 exits quietly."""
    env = {k: v for k, v in os.environ.items() if k not in ("WORLD_SIZE", "RANK", "LOCAL_RANK")}
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--impl", "reference",
                          "--workload", "C1", "--steps", "1", "--warmup", "0"], capture_output=True, text=True,
                         cwd=ROOT, env=env, timeout=600)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [json.loads(l) for l in out.stdout.strip().splitlines() if l.startswith("{")]
    assert len(lines) == 1 and lines[0]["impl"] == "reference" and lines[0]["n_gpus"] == 2
