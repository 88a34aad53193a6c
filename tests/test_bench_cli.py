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
        # taken on the kernel sources as they are now: a later edit of csrc/ or the header must come with new captures
        assert blk["stale"] is False, (path, blk.get("csrc_hash"), blk["bench_csrc_hash"])
        assert 0 < blk["hbm_frac"] < 0.2


import pytest


def _full_result_like_round_2():
    """A full result dict of the size that broke round 2 (its 27.9 KB one-line JSON overflowed the driver's 3 KB
    tail): the tracked detail of a default run, which has every leg, histogram and ncu summary."""
    import bench
    full = json.load(open(os.path.join(ROOT, "profiles", "r03_bench_pod.json")))
    full["roofline"]["ncu"] = bench._ncu_block(bench.NCU_POD)     # as a run of today's bench.py embeds it
    return full


def test_contract_line_fits_the_drivers_tail_and_keeps_the_contract_keys():
    import bench
    full = _full_result_like_round_2()
    assert len(json.dumps(full)) > 20000                    # the input really is the oversized one
    line = bench.compact_line(full, os.path.join(ROOT, "bench_detail.json"))
    text = json.dumps(line)
    assert len(text.encode()) <= bench.LINE_BUDGET == 3000, len(text)
    assert json.loads(text) == line
    for k in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
              "vs_baseline", "dtype", "data", "config", "e2e", "gpu_launches", "clocks", "roofline", "cpu_baseline",
              "kernel_ms", "variants", "aux", "sustained_ms", "detail"):
        assert k in line, k
    assert abs(line["value"] / full["value"] - 1) < 1e-4 and abs(line["ms_per_step"] / full["ms_per_step"] - 1) < 1e-4
    assert line["e2e"]["h2d_bytes_per_step"] == full["e2e"]["h2d_bytes_per_step"] and line["e2e"]["value"] > 0
    assert line["cpu_baseline"]["value"] > 0 and line["cpu_baseline"]["kind"] == "oracle"
    r = line["roofline"]
    assert r["bound"] == "alu" and r["kernel"] == "place_dense_kernel" and 0 < r["frac"] < 1 and r["peak"] > 0
    assert 0 < r["hbm_frac"] < 0.1 and r["warp_instr_per_request"] > 100 and r["issue_active_pct"] > 0
    assert set(line["variants"]) == {"dynamic_power_x4", "cold_starts_feasible", "ties", "identical_gpus"}
    assert set(line["aux"]) == {"local", "consol", "tiny", "rack"} and all(v["ok"] for v in line["aux"].values())
    assert len(line["config"]["workload"]) <= 200 and "configs[2]" in line["config"]["workload"]


def test_a_failed_extra_leg_is_reported_and_the_line_still_fits():
    import bench
    full = _full_result_like_round_2()
    full["aux"]["local"] = {"ok": False, "error": "AssertionError('CUDA and oracle disagree')" * 20}
    line = bench.compact_line(full)
    assert line["aux"]["local"]["ok"] is False and len(line["aux"]["local"]["error"]) <= 80
    assert len(json.dumps(line).encode()) <= bench.LINE_BUDGET


def test_ncu_block_reports_the_hbm_fraction_and_staleness():
    import bench
    blk = bench._ncu_block(bench.NCU_POD)
    peak = float(bench._peaks()[0].get("hbm_gbs", 6650.0))
    assert abs(blk["hbm_gbs"] - blk["dram_bytes"] / blk["duration_ns"]) < 1e-9 and abs(blk["hbm_frac"] - blk["hbm_gbs"] / peak) < 1e-12
    assert blk["bench_csrc_hash"] == bench._csrc_hash() and len(blk["bench_csrc_hash"]) == 12
    assert blk["stale"] in (True, False, None)
    if blk.get("csrc_hash"):
        assert blk["stale"] == (blk["csrc_hash"] != blk["bench_csrc_hash"])


def _run_bench(extra, timeout=1500):
    detail = os.path.join(ROOT, "gpurun_out", "test_bench_detail.json")
    os.makedirs(os.path.dirname(detail), exist_ok=True)
    p = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--steps", "3", "--warmup", "3", "--detail-out", detail] + extra,
                       capture_output=True, text=True, timeout=timeout)
    assert p.returncode == 0, p.stderr[-3000:]
    lines = [l for l in p.stdout.splitlines() if l.strip()]
    return lines, json.load(open(detail))


@pytest.mark.gpu
def test_default_invocation_ends_with_a_parseable_contract_line():
    """The DEFAULT run (variants and aux legs on, as the driver runs it): the headline line is printed before the
    extra legs, the enriched one last; every stdout line parses and fits the driver's 3 KB tail."""
    lines, detail = _run_bench([])
    assert len(lines) == 2, [l[:80] for l in lines]
    first, last = (json.loads(l) for l in lines)
    for l in lines:
        assert len(l.encode()) <= 3000, len(l)
    for d in (first, last):
        assert d["roofline"]["frac"] > 0 and d["cpu_baseline"]["value"] > 0 and d["e2e"]["value"] > 0 and d["value"] > 0
    assert "variants" not in first and first["value"] == last["value"] and first["ms_per_step"] == last["ms_per_step"]
    assert set(last["aux"]) == {"local", "consol", "tiny", "rack"} and len(last["variants"]) == 4
    assert all(v["ok"] for v in last["aux"].values()) and all(v["ok"] for v in last["variants"].values())
    assert len(detail["degeneracy"]["hist_phi"]) == 64 and "place_stats" in detail and "aux" in detail


@pytest.mark.gpu
def test_default_arm_prints_one_json_line_with_the_contract_keys():
    """A short run of the product arm on the GPU without the extra legs: ONE contract line on stdout, the full
    result (histograms, work counters) in the detail file."""
    lines, full = _run_bench(["--variants", "0", "--aux", "0", "--sustained-s", "0.2", "--cpu-requests", "256"], 900)
    assert len(lines) == 1, lines[:3]
    d = json.loads(lines[0])
    for k in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
              "vs_baseline", "dtype", "data", "config", "e2e", "gpu_launches", "clocks", "roofline", "cpu_baseline",
              "graph", "sustained_ms", "kernel_ms", "detail"):
        assert k in d, k
    for k in ("degeneracy", "place_stats", "sustained", "local_shape"):
        assert k in full, k
    assert d["n_gpus"] == 1 and d["steps"] == 3 and d["warmup"] == 3 and d["dtype"] == "f32" and d["data"] == "synthetic"
    assert d["value"] > 0 and d["ms_per_step"] > 0 and d["gpu_launches"] > 0 and d["vs_baseline"] is None
    assert "configs[2]" in d["config"]["workload"] and "workload" in d["config"]
    e = d["e2e"]
    assert e["value"] > 0 and e["h2d_bytes_per_step"] == 1024 * 128 + 65536 * 32 and e["d2h_bytes_per_step"] == 65536 * 32 + 1024 * 48
    assert e["value"] < d["value"]                       # the copies are inside the end-to-end timed region
    r = d["roofline"]
    assert r["bound"] == "alu" and 0 < r["frac"] < 1 and r["peak"] > 0 and abs(r["frac"] - r["achieved"] / r["peak"]) < 1e-3
    assert r["traffic"] is None or r["traffic"] > 0
    rf = full["roofline"]
    assert abs(rf["frac"] - rf["algorithmic_lane_ops_per_launch"] / (rf["kernel_ms"] * 1e-3) / (rf["peak"] * 1e12)) < 1e-9
    c = d["cpu_baseline"]
    assert c["kind"] == "oracle" and c["cores"] >= 1 and c["unit"] == d["unit"] and c["value"] > 0
    assert set(d["clocks"]) >= {"sm_mhz", "sm_max_mhz", "reasons"}
    g = full["degeneracy"]
    assert len(g["hist_phi"]) == 64 and len(g["hist_sigma"]) == 16 and len(g["hist_beta"]) == 128
