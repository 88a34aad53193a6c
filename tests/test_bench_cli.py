"""Host-side logic of bench.py that needs no GPU: the N-rank launch line, the reference arm's JSON contract and
the ncu summaries the roofline blocks quote."""
from __future__ import annotations

import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def test_gpus_n_starts_one_rank_per_gpu_on_localhost():
    import bench
    cmd = bench._spawn_cmd(4, ["--gpus", "4", "--steps", "3"])
    assert cmd[1:3] == ["-m", "torch.distributed.run"] and "--nproc-per-node=4" in cmd and "--nnodes=1" in cmd
    assert cmd[cmd.index("--master-addr") + 1] == "127.0.0.1" and 1024 < int(cmd[cmd.index("--master-port") + 1]) < 65536
    i = cmd.index(os.path.join(ROOT, "bench.py"))
    assert cmd[i + 1:] == ["--gpus", "4", "--steps", "3"]


def test_reference_arm_prints_one_json_line_with_the_contract_keys():
    p = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", "1", "--warmup", "0",
                        "--ref-requests", "32"], capture_output=True, text=True, timeout=600)
    assert p.returncode == 0, p.stderr[-2000:]
    lines = [l for l in p.stdout.splitlines() if l.strip()]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["gpu_launches"] == 0 and d["higher_is_better"] is True
    assert d["metric"] == "placement_candidate_evals_per_sec" and d["value"] > 0 and d["unit"] == d["cpu_baseline"]["unit"]
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["cores"] >= 1
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["e2e"]["d2h_bytes_per_step"] == 0
    assert "configs[2]" in d["config"]["workload"]


def test_tracked_ncu_summaries_are_what_the_roofline_blocks_read():
    import bench
    for path, kernel in ((bench.NCU_POD, "place_dense_kernel"), (bench.NCU_LOCAL, "local_slot_grouped_kernel"),
                         (bench.NCU_CONSOL, "consol_pair_kernel")):
        blk = bench._ncu_block(path)
        assert not blk.get("missing"), path
        assert kernel in blk["kernel"] and blk["warp_instructions"] > 0 and blk["duration_ns"] > 0
        assert blk["command"].startswith("ncu ") and blk["captured_at_git_sha"]


import pytest


@pytest.mark.gpu
def test_default_arm_prints_one_json_line_with_the_contract_keys():
    """A short run of the product arm on the GPU: one JSON line on stdout carrying the driver's contract keys."""
    p = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--steps", "3", "--warmup", "3", "--variants", "0",
                        "--aux", "0", "--sustained-s", "0.2", "--cpu-requests", "256"], capture_output=True, text=True, timeout=900)
    assert p.returncode == 0, p.stderr[-3000:]
    lines = [l for l in p.stdout.splitlines() if l.strip()]
    assert len(lines) == 1, lines[:3]
    d = json.loads(lines[0])
    for k in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
              "vs_baseline", "dtype", "data", "config", "e2e", "gpu_launches", "clocks", "roofline", "cpu_baseline",
              "graph", "sustained", "degeneracy", "place_stats", "kernel_ms"):
        assert k in d, k
    assert d["n_gpus"] == 1 and d["steps"] == 3 and d["warmup"] == 3 and d["dtype"] == "f32" and d["data"] == "synthetic"
    assert d["value"] > 0 and d["ms_per_step"] > 0 and d["gpu_launches"] > 0 and d["vs_baseline"] is None
    assert "configs[2]" in d["config"]["workload"] and "workload" in d["config"]
    e = d["e2e"]
    assert e["value"] > 0 and e["h2d_bytes_per_step"] == 1024 * 128 + 65536 * 32 and e["d2h_bytes_per_step"] == 65536 * 32 + 1024 * 48
    assert e["value"] < d["value"]                       # the copies are inside the end-to-end timed region
    r = d["roofline"]
    assert r["bound"] == "alu" and 0 < r["frac"] < 1 and r["peak"] > 0 and abs(r["frac"] - r["achieved"] / r["peak"]) < 1e-9
    assert r["traffic"] is None or r["traffic"] > 0
    c = d["cpu_baseline"]
    assert c["kind"] == "oracle" and c["cores"] >= 1 and c["unit"] == d["unit"] and c["value"] > 0
    assert set(d["clocks"]) >= {"sm_mhz", "sm_max_mhz", "reasons"}
    assert len(d["degeneracy"]["hist_phi"]) == 64 and len(d["degeneracy"]["hist_sigma"]) == 16 and len(d["degeneracy"]["hist_beta"]) == 128
