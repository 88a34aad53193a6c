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
