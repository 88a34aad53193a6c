#!/usr/bin/env python
"""bench.py — whole-hot-path throughput of libfestina_eval on N B200s (one process per GPU).

A *step* is one pass of the hot path over one batch of synthetic input (BASELINE.json
configs[2], "pod": K=1,024 GPUs, M=64 models, F=64, S=16, B=128, R=65,536 requests):
    fs_set_gpu_state (co-resident summaries)  ->  fs_place_batch (R requests)
    ->  fs_local_config on every GPU.
`value` = ELIGIBLE placement candidates of all ranks (every eligible (request, GPU) pair x its free shares x
F: the candidate set of the dense definition, what the CPU oracle evaluates one by one) / device time of the
step, inputs resident in HBM; the nominal grid R*K*S*F and what the kernel executed after exact pruning are
reported beside it.  `e2e` = the same through the C ABI with pinned HOST buffers (H2D of state + requests,
D2H of placements + local configs inside the timed region).
The default run (N = 1) then adds, outside the pod leg's timed region: `sustained` (seconds of back-to-back
replays), `variants` (pod reshaped so that pruning has less or nothing to hold on to), and `aux` (configs[3]
local sweep, configs[4] consolidation, configs[0]/[1] step times), each checked against the oracle in the run.
N > 1 (`--gpus N` starts N ranks itself through torch.distributed.run when not already under it): tables and
GPU state are replicated, every rank scores its own R requests (weak scaling, no data-path collective;
DESIGN.md "Multi-GPU"); the placement records are all-gathered over NCCL and rank 0 checks them.
`--impl reference` times the CPU oracle (test infrastructure) on a bounded sample instead.
`--ncu-import X.ncu-rep --ncu-out profiles/Y.json` turns an ncu capture into the small tracked summary the
roofline block quotes (no GPU needed).
"""
from __future__ import annotations

import argparse
import csv
import json
import math
import os
import socket
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from paper_2606_30391_b200 import synth  # noqa: E402
import bench_work  # noqa: E402

METRIC = "placement_candidate_evals_per_sec"
UNIT = "eligible candidates/s"
# DESIGN.md §7 "Roofline": lane-operations (one 32-bit load / arithmetic / compare / select on one
# lane) the method needs per unit of work, for the units the scoring kernel counts itself
OPS_PER_CANDIDATE = 13.0   # dense definition: 8 fp32 arithmetic + 5 compare/select
OPS_REQUEST = 96.0         # per request: two 16-byte plane-minima records per share lane, three bounds (32 lanes x 3)
OPS_TILE = 12.0            # per (request, sigma, phi) of a built tile: 4 table values, 5 fp32, test + select, running minimum
OPS_PAIR_TEST = 18.0       # per (request, GPU) tested: 8-word record, 7 eligibility compares, bound (2 fp32 + compare)
OPS_TSTAR = 12.0           # per swept pair: deadline threshold T*
OPS_SWEEP = 2.0            # per swept candidate: compare + predicated min
OPS_ROW = 4.0              # per swept (pair, phi): A0 load, add, min, subtract/compare share
OPS_WARM_TEST = 30.0       # per warm pair tested: 16-word item, bound (2 table bounds + 4 fp32), 3 compares
OPS_DEF = 15.0             # per candidate scored by the definition: 4 loads, 4 mul, 4 add/sub, 3 compares
SM_COUNT, ISSUE_LANES_PER_CLK_PER_SM = 148, 128   # 4 schedulers x 32 lanes (B300_MICROARCH "issue")
NCU_POD = os.path.join(ROOT, "profiles", "r03_pod_ncu.json")
NCU_LOCAL = os.path.join(ROOT, "profiles", "r03_local_ncu.json")
NCU_CONSOL = os.path.join(ROOT, "profiles", "r03_consol_ncu.json")


def _peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return json.load(open(p)), "measured"
        except Exception:
            pass
    return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0}, "fallback"


def _alu_peak():
    peaks, src = _peaks()
    mhz = float(peaks.get("sm_max_mhz", 1965.0))
    return SM_COUNT * ISSUE_LANES_PER_CLK_PER_SM * mhz * 1e6, mhz, src


def _git_sha():
    try:
        sha = subprocess.run(["git", "rev-parse", "--short", "HEAD"], cwd=ROOT, capture_output=True, text=True).stdout.strip()
        return sha or None
    except OSError:
        return None


def _csrc_hash():
    """sha1 over the kernel sources and the header (names and bytes): what an ncu capture is a capture OF.  Works
    on the GPU box, where the snapshot has no .git."""
    import glob
    import hashlib
    h = hashlib.sha1()
    files = sorted(glob.glob(os.path.join(ROOT, "paper_2606_30391_b200", "csrc", "*"))) + [os.path.join(ROOT, "include", "festina_eval.h")]
    for f in files:
        h.update(os.path.basename(f).encode()); h.update(open(f, "rb").read())
    return h.hexdigest()[:12]


def _ncu_block(path):
    """The tracked summary of an ncu capture (written by --ncu-import) with the hash of the sources it was taken
    on beside the hash of the sources now, so that a stale capture shows (`stale`: true / false, None when the
    summary predates the hash): the figures are evidence from a profiler run, never measured inside the bench."""
    if not os.path.exists(path):
        return {"source": os.path.relpath(path, ROOT), "missing": True}
    d = json.load(open(path))
    d["source"] = os.path.relpath(path, ROOT)
    d["bench_git_sha"] = _git_sha()
    d["bench_csrc_hash"] = _csrc_hash()
    d["stale"] = (d["csrc_hash"] != d["bench_csrc_hash"]) if d.get("csrc_hash") else None
    if d.get("dram_bytes") and d.get("duration_ns"):
        d["hbm_gbs"] = d["dram_bytes"] / d["duration_ns"]
        d["hbm_frac"] = d["hbm_gbs"] / float(_peaks()[0].get("hbm_gbs", 6650.0))
    return d


LINE_BUDGET = 3000   # bytes: the driver keeps a 3 KB tail of stdout, the contract line has to fit in it


def _r(x, n=5):
    """Floats to n significant digits (the line has a byte budget); everything else unchanged."""
    if isinstance(x, float) and math.isfinite(x):
        return float(f"{x:.{n}g}")
    return x


def _roofline_scalars(rf, requests=None):
    ncu = rf.get("ncu") or {}
    out = {"bound": rf.get("bound"), "kernel": str(rf.get("kernel", "")).split(" ")[0], "achieved": _r(rf.get("achieved")),
           "peak": _r(rf.get("peak")), "unit": rf.get("unit"), "frac": _r(rf.get("frac")), "traffic": rf.get("traffic"),
           "kernel_ms": _r(rf.get("kernel_ms"))}
    if "survey_formula" in rf:
        out["survey_formula_frac"] = _r(rf["survey_formula"].get("frac"))
    if "sweep_pipe" in rf:
        out["sweep_pipe_frac"] = _r(rf["sweep_pipe"].get("frac"))
    if ncu and not ncu.get("missing"):
        out.update({"hbm_frac": _r(ncu.get("hbm_frac")), "hbm_gbs": _r(ncu.get("hbm_gbs")),
                    "issue_active_pct": _r(ncu.get("issue_active_pct")), "ncu": ncu.get("source"),
                    "ncu_csrc_hash": ncu.get("csrc_hash"), "ncu_stale": ncu.get("stale")})
        if requests and ncu.get("warp_instructions"):
            out["warp_instr_per_request"] = _r(ncu["warp_instructions"] / requests)
    return out


def compact_line(full: dict, detail_path=None) -> dict:
    """The contract line the driver parses (at most LINE_BUDGET bytes as JSON): the contract keys, `roofline`,
    `cpu_baseline`, `e2e`, `clocks` and one scalar triple per extra leg.  Histograms, work counters, notes and
    the whole ncu summaries stay in the detail file (`detail`)."""
    cfg = dict(full.get("config", {}))
    cfg["workload"] = str(cfg.get("workload", ""))[:200]
    for k in ("l2", "parallelism"):
        if k in cfg:
            cfg[k] = str(cfg[k])[:60]
    line = {k: _r(full.get(k)) for k in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step",
                                         "higher_is_better", "scaling", "vs_baseline", "dtype", "data", "gpu_launches")}
    line["config"] = cfg
    ck = full.get("clocks") or {}
    line["clocks"] = {k: ck.get(k) for k in ("sm_mhz", "sm_max_mhz", "reasons")}
    e = full.get("e2e") or {}
    line["e2e"] = {k: _r(e.get(k)) for k in ("value", "unit", "ms_per_step", "h2d_bytes_per_step", "d2h_bytes_per_step")}
    if "cpu_baseline" in full:
        c = full["cpu_baseline"]
        line["cpu_baseline"] = {"value": _r(c.get("value")), "unit": c.get("unit"), "cores": c.get("cores"),
                                "kind": c.get("kind"), "sample": str(c.get("sample", ""))[:120]}
    line["kernel_ms"] = {k: _r(v, 4) for k, v in (full.get("kernel_ms") or {}).items()}
    if "roofline" in full:
        line["roofline"] = _roofline_scalars(full["roofline"], (full.get("place_stats") or {}).get("requests"))
    g = full.get("graph")
    line["graph"] = bool(g.get("device_step")) if isinstance(g, dict) else bool(g)
    if "sustained" in full:
        line["sustained_ms"] = _r(full["sustained"].get("ms_per_step"))
    if "gathered_records_ok" in full:
        line["gathered_records_ok"] = full["gathered_records_ok"]

    def triple(leg, ms_key):
        if not isinstance(leg, dict):
            return {"ok": False}
        if leg.get("ok") is False:
            return {"ok": False, "error": str(leg.get("error", ""))[:80]}
        t = {"ms": _r(leg.get(ms_key, leg.get("ms_per_step")), 4), "ok": True}
        if "roofline" in leg:
            t["frac"] = _r(leg["roofline"].get("frac"), 4)
        return t
    if "variants" in full:
        line["variants"] = {k: triple(v, "place_score_ms") for k, v in full["variants"].items()}
    if "aux" in full:
        line["aux"] = {k: triple(v, "ms_per_step") for k, v in full["aux"].items()}
    if detail_path:
        line["detail"] = os.path.relpath(detail_path, ROOT) if os.path.isabs(detail_path) else detail_path
    return line


def emit(full: dict, detail_path=None):
    """Write the full result to the detail file and print the contract line (one line, flushed)."""
    if detail_path:
        try:
            json.dump(full, open(detail_path, "w"), indent=1)
        except OSError as e:
            print(f"bench.py: could not write {detail_path}: {e}", file=sys.stderr)
            detail_path = None
    text = json.dumps(compact_line(full, detail_path))
    assert len(text.encode()) <= LINE_BUDGET, f"contract line is {len(text.encode())} bytes (budget {LINE_BUDGET})"
    print(text, flush=True)


class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int, period_ms: int = 100):
        self.rows, self.proc, self.thr = [], None, None
        self.cmd = ["nvidia-smi", f"--id={index}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                    "-lms", str(period_ms)]

    def start(self):
        try:
            self.proc = subprocess.Popen(self.cmd, stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except OSError:
            return self

        def pump():
            for line in self.proc.stdout:
                self.rows.append([x.strip() for x in line.split(",")])
        self.thr = threading.Thread(target=pump, daemon=True)
        self.thr.start()
        return self

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, reasons, pw = [], [], set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            if len(r) < 7:
                continue
            try:
                sm.append(float(r[0])); mx.append(float(r[1])); pw.append(float(r[2]))
            except ValueError:
                continue
            for n, v in zip(names, r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


def _dist():
    ws = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    lrank = int(os.environ.get("LOCAL_RANK", "0"))
    return ws, rank, lrank


def _hist(a, n):
    """Counts of the values 0..n-1 of an integer array (the chosen-index histograms of SURVEY 8(d))."""
    a = np.asarray(a).reshape(-1)
    a = a[(a >= 0) & (a < n)]
    return np.bincount(a.astype(np.int64), minlength=n).astype(int).tolist()


def _top_share(h):
    t = sum(h)
    return float(max(h) / t) if t else 0.0


WORKLOAD_CFG = {"tiny": "configs[0]", "rack": "configs[1]", "pod": "configs[2]", "local": "configs[3]", "consol": "configs[4]"}


def _workload_name(cl):
    base = cl.name.split("/")[0]
    tag = f"BASELINE.json {WORKLOAD_CFG[base]}" if base in WORKLOAD_CFG else "custom"
    return f"{cl.name} ({tag})"


def _config(cl, args, ws, graph):
    return {"workload": f"{_workload_name(cl)}: K={cl.K} GPUs, M={cl.M}, F={cl.F}, S={cl.S}, "
                        f"B={cl.B}, R={cl.R} requests per rank; step = fs_set_gpu_state + fs_place_batch + "
                        f"fs_local_config(all GPUs, energy objective, exhaustive splits"
                        + (", then the minimum-SM split rule" if args.split_modes == "both" else "") + ")"
                        + ("; the two calls on two streams" if args.overlap else "")
                        + ("; one CUDA graph per step" if graph else ""),
            "K": cl.K, "M": cl.M, "F": cl.F, "S": cl.S, "B": cl.B, "R_per_rank": cl.R,
            "l2": "flushed between timed steps by overwriting a 256 MiB buffer",
            "parallelism": f"replicated tables+state, requests sharded x{ws}"}


def oracle_sample(cl, n_req: int, nthreads: int):
    """One bounded pass of the hot path through the CPU oracle; returns (seconds, eligible candidates, GPUs)."""
    import oracle
    n_gpu = max(1, int(round(cl.K * n_req / max(cl.R, 1))))
    reqs = cl.requests[:n_req]
    t0 = time.perf_counter()
    oracle.place_batch(cl.lat, cl.pow, cl.models, cl.states, reqs, nthreads)
    oracle.local_config(cl.lat, cl.pow, cl.states, 0, np.arange(n_gpu, dtype=np.int32), nthreads)
    dt = time.perf_counter() - t0
    return dt, bench_work.eligible_work(cl, reqs)[1], n_gpu


def run_reference(args):
    ws, rank, _ = _dist()
    if rank != 0:
        return
    cl = synth.make_cluster(args.workload if args.workload in ("tiny", "rack", "pod") else "pod")
    cores = os.cpu_count() or 1
    n_req = min(args.ref_requests, cl.R)
    for _ in range(args.warmup):
        oracle_sample(cl, max(8, n_req // 8), cores)
    tot, cand, n_gpu = 0.0, 0, 0
    for _ in range(args.steps):
        dt, c, n_gpu = oracle_sample(cl, n_req, cores)
        tot += dt; cand += c
    val = cand / tot
    sample = (f"{n_req} of {cl.R} requests x all {cl.K} GPUs (fs_place_batch) + {n_gpu} GPUs "
              f"(fs_local_config) per step")
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * tot / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32",
            "data": "synthetic", "config": _config(cl, args, args.gpus, False),
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def _place_shape(cl, place):
    """What the decisions look like (histograms of the chosen indices in every run)."""
    ok = place["gpu"] >= 0
    hp, hs, hb = _hist(place["phi"][ok], cl.F), _hist(place["sigma"][ok], cl.S), _hist(place["beta"][ok], cl.B)
    return {"placed_frac": float(ok.mean()) if len(ok) else 0.0, "top_phi_share": _top_share(hp),
            "top_sigma_share": _top_share(hs), "top_beta_share": _top_share(hb),
            "distinct_gpus": int(len(np.unique(place["gpu"][ok]))),
            "hist_phi": hp, "hist_sigma": hs, "hist_beta": hb}


def _local_shape(cl, res):
    ok = res["phi"] >= 0
    live = np.arange(4)[None, :] < cl.states["n_res"][: len(res), None]
    sel = ok[:, None] & live
    hp = _hist(res["phi"][ok], cl.F)
    hs = _hist(res["sigma"][sel], cl.S)
    busy = cl.states["t"]["q"][: len(res)] > 0
    hb = _hist(res["beta"][sel[:, :, None] & busy], cl.B)
    return {"feasible_frac": float(ok.mean()) if len(ok) else 0.0, "top_phi_share": _top_share(hp),
            "top_sigma_share": _top_share(hs), "top_beta_share": _top_share(hb),
            "hist_phi": hp, "hist_sigma": hs, "hist_beta": hb}


def _useful_ops(cl, ps):
    """Lane-operations of the units the scoring kernel counted itself (DESIGN.md section 7 per-unit figures)."""
    return (OPS_REQUEST * ps["requests"] + OPS_TILE * ps["tiles_built"] * cl.S * cl.F
            + OPS_PAIR_TEST * 32 * ps["chunks_tested"] + OPS_TSTAR * ps["cold_pairs_swept"]
            + OPS_SWEEP * ps["cold_candidates_swept"] + OPS_ROW * cl.F * ps["cold_pairs_swept"]
            + OPS_WARM_TEST * ps["warm_pairs_tested"] + OPS_DEF * ps["candidates_scored"])


def _place_roofline(cl, ps, score_ms, cand_def, ncu_path=None):
    alu_peak, mhz, peak_src = _alu_peak()
    useful = _useful_ops(cl, ps)
    executed = ps["cold_candidates_swept"] + ps["candidates_scored"]
    # frac: the lane-ops of every unit the kernel counted itself, each weighted with what that unit costs (DESIGN.md
    # section 7: a swept candidate is a compare and a predicated min, a candidate scored by the definition 15, ...)
    # over the launch's CUDA-event time, against the issue peak.  SURVEY 8(d)'s flat 13 lane-ops x candidates
    # evaluated charges a swept candidate like a full evaluation (it exceeds 1 on sweep-dominated inputs): it is
    # kept beside it as survey_formula.
    survey = OPS_PER_CANDIDATE * executed
    achieved = useful / (score_ms * 1e-3)
    nominal = OPS_PER_CANDIDATE * cand_def / (score_ms * 1e-3)
    blk = {"bound": "alu", "kernel": "place_dense_kernel (fs_place_batch scoring + argmin + records)",
           "achieved": achieved / 1e12, "peak": alu_peak / 1e12, "unit": "Tlane-op/s", "frac": achieved / alu_peak,
           "traffic": None, "algorithmic_lane_ops_per_launch": useful, "kernel_ms": score_ms,
           "executed_candidates_per_launch": executed,
           "executed_frac_of_eligible": executed / cand_def if cand_def else None,
           "survey_formula": {"lane_ops_per_unit": OPS_PER_CANDIDATE, "lane_ops_per_launch": survey,
                              "achieved": survey / (score_ms * 1e-3) / 1e12, "frac": survey / (score_ms * 1e-3) / alu_peak,
                              "note": "13 lane-ops (SURVEY 8(d)) x candidates evaluated by this launch (swept + scored by the "
                                      "definition): over-counts swept candidates, above 1 on sweep-dominated inputs"},
           "dense_definition": {"achieved": nominal / 1e12, "frac": nominal / alu_peak,
                                "note": f"{OPS_PER_CANDIDATE:g} lane-ops x {cand_def} eligible candidates / kernel time; "
                                        "above 1 when exact pruning skips most of them: it measures the algorithm, not the kernel"},
           "note": "achieved = lane-ops of the units the kernel counted (requests, built tiles, records tested, swept pairs "
                   "and candidates, warm pairs tested, candidates scored by the definition; DESIGN.md section 7 per-unit "
                   "figures) / CUDA-event time of the launch; peak = 148 SMs x 128 lanes/clk x "
                   f"{mhz:.0f} MHz ({peak_src} sm_max_mhz)"}
    if ps["cold_candidates_swept"] > 4 * ps["candidates_scored"]:
        # sweep-dominated launch (the bounds cannot prune): the swept candidates against the rate at which an SM
        # issues the sweep's compare + predicated-min pair (profiles/r01_pipe_rates.md: 31.6 pairs per clock per SM)
        pair_peak = 31.6 * SM_COUNT * mhz * 1e6
        rate = ps["cold_candidates_swept"] / (score_ms * 1e-3)
        blk["sweep_pipe"] = {"achieved": rate / 1e12, "peak": pair_peak / 1e12, "unit": "Tcandidate/s", "frac": rate / pair_peak,
                             "note": "swept candidates / kernel time against 31.6 compare+predicated-min pairs per clock per SM"}
    if ncu_path:
        ncu = _ncu_block(ncu_path)
        blk["ncu"] = ncu
        if not ncu.get("missing"):
            blk["traffic"] = ncu.get("dram_bytes")
            blk["hbm_frac"] = ncu.get("hbm_frac")
            wi = ncu.get("warp_instructions")
            if wi:
                blk["useful_per_issued"] = useful / 32.0 / wi
    return blk


def _tb(torch, dev, a):
    return torch.from_numpy(np.ascontiguousarray(a).view(np.uint8).reshape(-1)).to(dev)


def _capture(torch, dev, stream, fn, what):
    """One CUDA graph of fn(stream); None (and a note on stderr) when capture fails: the JSON line says which
    path was timed ("graph": true | false), so a direct-launch number is never mistaken for the graph path."""
    try:
        cap = torch.cuda.Stream(device=dev)
        cap.wait_stream(stream)
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=cap):
            fn(torch.cuda.current_stream())
        stream.wait_stream(cap)
        for _ in range(3):
            g.replay()
        torch.cuda.synchronize()
        return g
    except Exception as e:                              # noqa: BLE001 - reported, and the fallback is flagged
        print(f"bench.py: CUDA graph capture of {what} failed ({e}); timing direct launches", file=sys.stderr)
        torch.cuda.synchronize()
        return None


def run_ours(args):
    import torch
    import paper_2606_30391_b200 as fs

    ws, rank, lrank = _dist()
    dist = None
    if ws > 1 or "TORCHELASTIC_RUN_ID" in os.environ:   # under torch.distributed.run, also with a single rank
        import torch.distributed as dist
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("NCCL_DEBUG", "INFO")     # the communicator lines (nranks, NVLS) ...
        os.environ.setdefault("NCCL_DEBUG_FILE", "/dev/stderr")   # ... on stderr: stdout carries the one JSON line
        torch.cuda.set_device(lrank)
        dist.init_process_group("nccl", device_id=torch.device("cuda", lrank))
    dev = torch.device("cuda", lrank)
    torch.cuda.set_device(dev)
    cl = synth.make_cluster(args.workload)
    if rank > 0:   # every rank scores its own batch
        cl.requests = synth.make_requests(cl.seed + 7919 * rank, cl.R, cl.M)
    ctx = fs.Festina(lrank)
    tb = lambda a: _tb(torch, dev, a)
    # offline profile tables are loaded once (profiling is offline), not per step
    ctx.load_profiles(torch.from_numpy(cl.lat).to(dev), torch.from_numpy(cl.pow).to(dev), tb(cl.freq_mhz),
                      tb(cl.models), cl.params)
    d_states, d_reqs = tb(cl.states), tb(cl.requests)
    d_place = torch.empty(cl.R * 32, dtype=torch.uint8, device=dev)
    d_local = torch.empty(cl.K * 48, dtype=torch.uint8, device=dev)
    both_splits = args.split_modes == "both"
    d_local2 = torch.empty(cl.K * 48, dtype=torch.uint8, device=dev)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    stream = torch.cuda.current_stream()
    ctx.set_timing(True)

    # fs_place_batch and fs_local_config both depend only on the state: the step issues them on two
    # streams so that the slot search fills the issue slots the placement kernel leaves (same host thread)
    side = torch.cuda.Stream(device=dev) if args.overlap else None
    ev_state, ev_side = torch.cuda.Event(), torch.cuda.Event()

    def step(states, reqs, place, local, local2, pinned, serial=False, st=None):
        st = stream if st is None else st
        ctx.set_gpu_state(states, stream=st, pinned=pinned)
        if side is None or serial:
            ctx.place_batch(reqs, out=place, stream=st, pinned=pinned)
            ctx.local_config(0, n=cl.K, out=local, stream=st, pinned=pinned)
            if both_splits:
                ctx.local_config(2, n=cl.K, out=local2, stream=st, pinned=pinned)
            return
        ev_state.record(st)
        side.wait_event(ev_state)
        ctx.local_config(0, n=cl.K, out=local, stream=side, pinned=pinned)
        if both_splits:
            ctx.local_config(2, n=cl.K, out=local2, stream=side, pinned=pinned)
        ctx.place_batch(reqs, out=place, stream=st, pinned=pinned)
        ev_side.record(side)
        st.wait_event(ev_side)

    def step_device(serial=False, st=None):
        step(d_states, d_reqs, d_place, d_local, d_local2, False, serial, st)

    def barrier():
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
            torch.cuda.synchronize()

    warm = max(args.warmup, 3)
    for _ in range(warm):
        step_device()
    barrier()
    # The calls are asynchronous and allocation-free after the first step, so a whole step (fork to the second
    # stream and join included) can be captured into a CUDA graph and replayed: one launch per step for the host.
    graph, launches_per_step = None, None
    lc = ctx.launch_count
    step_device()
    launches_per_step = ctx.launch_count - lc
    torch.cuda.synchronize()
    if args.graph:
        ctx.set_timing(False)                           # event records of the per-kernel timers are not capturable
        graph = _capture(torch, dev, stream, lambda st: step_device(st=st), "the device step")
        ctx.set_timing(True)
    barrier()
    sampler = ClockSampler(lrank).start()
    evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    kt = {}
    barrier()
    wall0 = time.perf_counter()
    for a, b in evs:
        flush.zero_()                      # L2 flush, outside the per-step events
        a.record(stream)
        if graph is not None:
            graph.replay()
        else:
            step_device()
        b.record(stream)
        b.synchronize()
        if side is None and graph is None:
            for k, v in ctx.get_timing().items():
                kt.setdefault(k, []).append(v)
    barrier()
    wall = time.perf_counter() - wall0
    launches = launches_per_step * args.steps
    dev_ms = sum(a.elapsed_time(b) for a, b in evs)
    # per-kernel durations need the kernels one after the other: when the timed steps overlap the two calls,
    # the same K steps are run once more serially (same inputs, L2 flushed) for kernel_ms and the roofline
    serial_ms = dev_ms
    if side is not None or graph is not None:
        serial_ms = 0.0
        for _ in range(args.steps):
            flush.zero_()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(stream); step_device(serial=True); b.record(stream); b.synchronize()
            serial_ms += a.elapsed_time(b)
            for k, v in ctx.get_timing().items():
                kt.setdefault(k, []).append(v)
    # work counters: one untimed call with the kernel's counters switched on (same input, same work)
    ctx.set_work_stats(True)
    ctx.place_batch(d_reqs, out=d_place, stream=stream)
    pstats = ctx.last_place_stats()
    ctx.set_work_stats(False)
    pairs, cand_def = bench_work.eligible_work(cl)

    # ---- sustained: seconds of back-to-back replays, no flush, clocks sampled over that window ----------
    sustained = None
    if rank == 0 and args.sustained_s > 0:
        n_rep = max(50, int(math.ceil(args.sustained_s * 1e3 / max(dev_ms / args.steps, 1e-3))))
        s2 = ClockSampler(lrank, 50).start()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(stream)
        for _ in range(n_rep):
            if graph is not None:
                graph.replay()
            else:
                step_device()
        b.record(stream); b.synchronize()
        sus_ms = a.elapsed_time(b)
        sustained = {"steps": n_rep, "seconds": sus_ms * 1e-3, "ms_per_step": sus_ms / n_rep,
                     "value": cand_def * n_rep / (sus_ms * 1e-3), "unit": UNIT, "clocks": s2.stop(),
                     "note": "back-to-back " + ("graph replays" if graph is not None else "direct steps")
                             + " of the same step, no L2 flush in between (tables and state stay in the 126 MB L2)"}

    # ---- end to end through the C ABI with pinned host buffers --------------------------------------
    h_states = torch.from_numpy(cl.states.view(np.uint8).reshape(-1).copy()).pin_memory()
    h_reqs = torch.from_numpy(cl.requests.view(np.uint8).reshape(-1).copy()).pin_memory()
    h_place = torch.empty(cl.R * 32, dtype=torch.uint8).pin_memory()
    h_local = torch.empty(cl.K * 48, dtype=torch.uint8).pin_memory()
    h_local2 = torch.empty(cl.K * 48, dtype=torch.uint8).pin_memory()

    # The same step with FS_HOST_PINNED buffers: every step copies its inputs (state records, requests)
    # from page-locked host memory and its results (placements, local configurations) back; the host waits for
    # the stream before it reads them.  Two streams and one CUDA graph per step, as in the device-resident step.
    def step_host(st=None):
        step(h_states, h_reqs, h_place, h_local, h_local2, True, False, st)

    ctx.set_timing(False)
    for _ in range(3):
        step_host()
    torch.cuda.synchronize()
    hgraph = _capture(torch, dev, stream, lambda st: step_host(st=st), "the host-buffer step") if args.graph else None
    barrier()
    e2e_t = 0.0
    for _ in range(args.steps):
        flush.zero_()
        h_place.zero_()
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        if hgraph is not None:
            hgraph.replay()
        else:
            step_host()
        torch.cuda.synchronize()
        e2e_t += time.perf_counter() - t0
    clocks = sampler.stop()
    assert np.array_equal(h_place.numpy(), d_place.cpu().numpy()), "host and device paths disagree"
    assert np.array_equal(h_local.numpy(), d_local.cpu().numpy()), "host and device paths disagree (local)"

    # ---- N > 1: the placement records of all ranks, gathered on the device over NCCL; rank 0 recomputes
    # every rank's batch on its own GPU and compares the bytes
    gathered_ok = None
    if dist is not None:
        from paper_2606_30391_b200 import shard
        allrec = shard.gather_records(d_place, [cl.R] * ws, dist, dtype=synth.PLACEMENT_DT)
        if rank == 0:
            gathered_ok = len(allrec) == ws * cl.R
            d_chk = torch.empty_like(d_place)
            for r in range(ws):
                rq = cl.requests if r == 0 else synth.make_requests(cl.seed + 7919 * r, cl.R, cl.M)
                ctx.place_batch(tb(rq), out=d_chk, stream=stream)
                torch.cuda.synchronize()
                gathered_ok = gathered_ok and np.array_equal(d_chk.cpu().numpy().view(synth.PLACEMENT_DT),
                                                             allrec[r * cl.R:(r + 1) * cl.R])

    t = torch.tensor([dev_ms, e2e_t * 1e3, wall * 1e3], dtype=torch.float64, device=dev)
    if dist is not None:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dev_ms, e2e_ms, wall_ms = (float(x) for x in t.cpu())
    if rank != 0:
        ctx.close()
        if dist is not None:
            dist.destroy_process_group()
        return
    grid_cands = cl.R * cl.K * cl.S * cl.F
    steps = args.steps
    score_ms = float(np.mean(kt.get("place_score", [float("nan")])))
    place = d_place.cpu().numpy().view(synth.PLACEMENT_DT)
    local = d_local.cpu().numpy().view(synth.LOCAL_CFG_DT)
    line = {
        "metric": METRIC, "value": ws * cand_def * steps / (dev_ms * 1e-3), "unit": UNIT, "n_gpus": ws, "steps": steps,
        "warmup": warm, "ms_per_step": dev_ms / steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32", "data": "synthetic", "config": _config(cl, args, ws, graph is not None),
        "graph": {"device_step": graph is not None, "host_step": hgraph is not None},
        "decisions_per_sec": ws * (cl.R + cl.K) * steps / (dev_ms * 1e-3),
        "placement_decisions_per_sec": ws * cl.R * steps / (dev_ms * 1e-3),
        "nominal_grid_candidates_per_sec": ws * grid_cands * steps / (dev_ms * 1e-3),
        "executed_candidates_per_sec": ws * (pstats["cold_candidates_swept"] + pstats["candidates_scored"]) * steps / (dev_ms * 1e-3),
        "nominal_candidates_per_step": grid_cands, "eligible_candidates_per_step": cand_def,
        "eligible_pairs_per_step": pairs, "place_stats": pstats,
        "value_note": "value = eligible candidates (the dense definition's candidate set, what the oracle evaluates one by "
                      "one) / step time; the kernel reaches the same argmin after scoring executed_candidates of them "
                      "(exact branch and bound), so value measures the method on this workload, roofline.frac the kernel",
        "kernel_ms": {k: float(np.mean(v)) for k, v in kt.items()},
        "serial": {"ms_per_step": serial_ms / steps,
                   "note": ("timed steps run fs_place_batch and fs_local_config on two streams"
                            + (", replayed from one CUDA graph per step" if graph is not None else "")
                            + "; kernel_ms and the roofline come from the same steps run serially, launch by launch, "
                              "right after" if (args.overlap or graph is not None) else
                            "timed steps are serial: kernel_ms comes from them")},
        "wall_ms_per_step_incl_flush": wall_ms / steps,
        "e2e": {"value": ws * cand_def * steps / (e2e_ms * 1e-3), "unit": UNIT, "ms_per_step": e2e_ms / steps,
                "h2d_bytes_per_step": cl.K * 128 + cl.R * 32, "d2h_bytes_per_step": cl.R * 32 + cl.K * 48 * (2 if both_splits else 1),
                "mode": "FS_HOST_PINNED buffers (page-locked host memory): state records and local configurations by "
                        "copy engine, requests read and placement records written over PCIe by the scoring kernel itself"
                        + (", two streams" if side is not None else "") + (", one CUDA graph per step" if hgraph is not None else ", direct calls")
                        + "; host wall clock around the step incl. the final stream synchronisation"},
        "gpu_launches": int(launches),
        "clocks": clocks,
        "roofline": _place_roofline(cl, pstats, score_ms, cand_def, NCU_POD),
        "degeneracy": _place_shape(cl, place),
        "local_shape": _local_shape(cl, local),
    }
    if sustained is not None:
        line["sustained"] = sustained
    if gathered_ok is not None:
        line["gathered_records_ok"] = bool(gathered_ok)
        assert gathered_ok, "records gathered over NCCL differ from the recomputation on rank 0"
    detail = args.detail_out
    if ws == 1 and not args.no_cpu_baseline:
        cores = os.cpu_count() or 1
        dt, c, n_gpu = oracle_sample(cl, args.cpu_requests, cores)
        line["cpu_baseline"] = {"value": c / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
                                "sample": f"{args.cpu_requests} of {cl.R} requests x all {cl.K} GPUs + "
                                          f"{n_gpu} GPUs local config, {dt:.1f} s"}
    if ws == 1 and (args.variants or args.aux):
        # the headline first: whatever happens in an extra leg below, this line is already on stdout.  The
        # enriched line (same pod numbers + one triple per extra leg) is printed last.
        emit(line, detail)

        def guarded(fn, *a):
            try:
                return fn(*a)
            except Exception as e:                          # noqa: BLE001 - reported in the line and on stderr
                print(f"bench.py: leg {fn.__name__}{a[-2:-1]} failed: {e!r}", file=sys.stderr)
                return {"ok": False, "error": repr(e)}
        ctx.set_timing(True)
        if args.variants:
            line["variants"] = {n: guarded(run_variant, args, torch, dev, ctx, n, flush) for n in bench_work.VARIANTS}
        if args.aux:
            line["aux"] = {w: guarded(run_aux_leg, args, torch, dev, w, flush) for w in ("local", "consol")}
            line["aux"].update({w: guarded(run_small_leg, args, torch, dev, w, flush) for w in ("tiny", "rack")})
    emit(line, detail)
    ctx.close()
    if dist is not None:
        dist.destroy_process_group()


def run_variant(args, torch, dev, ctx, name, flush):
    """configs[2] reshaped so that the bounds prune less (or nothing): the scoring kernel timed on the variant, with
    its work counters, its roofline fraction and the shape of the decisions; checked against the oracle on a sample
    of its requests in this run."""
    import oracle
    stream = torch.cuda.current_stream()
    cores = os.cpu_count() or 1
    cl = bench_work.make_variant(args.workload, name)
    tb = lambda a: _tb(torch, dev, a)
    ctx.load_profiles(torch.from_numpy(cl.lat).to(dev), torch.from_numpy(cl.pow).to(dev), tb(cl.freq_mhz),
                      tb(cl.models), cl.params)
    d_states, d_reqs = tb(cl.states), tb(cl.requests)
    d_place = torch.empty(cl.R * 32, dtype=torch.uint8, device=dev)
    n_steps = max(3, args.steps // 2) if name != "identical_gpus" else 3
    ts, step_ms = [], []
    for i in range(3 + n_steps):
        flush.zero_()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(stream)
        ctx.set_gpu_state(d_states, stream=stream)
        ctx.place_batch(d_reqs, out=d_place, stream=stream)
        b.record(stream); b.synchronize()
        if i >= 3:
            ts.append(ctx.get_timing()["place_score"]); step_ms.append(a.elapsed_time(b))
    ctx.set_work_stats(True)
    ctx.place_batch(d_reqs, out=d_place, stream=stream)
    ps = ctx.last_place_stats()
    ctx.set_work_stats(False)
    place = d_place.cpu().numpy().view(synth.PLACEMENT_DT)
    idx = np.arange(0, cl.R, max(1, cl.R // args.variant_sample))
    ref = oracle.place_batch(cl.lat, cl.pow, cl.models, cl.states, cl.requests[idx], cores)
    same = all(np.array_equal(place[idx][f], ref[f]) for f in ("gpu", "sigma", "phi", "beta", "f_req", "flat")) and \
        np.array_equal(place[idx]["energy_mj"].view(np.uint32), ref["energy_mj"].view(np.uint32))
    assert same, f"variant {name}: CUDA and oracle disagree on the sample"
    pairs, cand_def = bench_work.eligible_work(cl)
    score_ms = float(np.mean(ts))
    shape = _place_shape(cl, place)
    for k in ("hist_sigma", "hist_beta"):
        shape.pop(k)
    return {"place_score_ms": score_ms, "ms_per_step": float(np.mean(step_ms)), "steps": n_steps,
            "step": "fs_set_gpu_state + fs_place_batch, L2 flushed between steps",
            "value": cand_def / (float(np.mean(step_ms)) * 1e-3), "unit": UNIT,
            "eligible_candidates_per_step": cand_def, "place_stats": ps,
            "roofline": _place_roofline(cl, ps, score_ms, cand_def),
            "degeneracy": shape,
            "oracle_check": f"{len(idx)} requests (every {max(1, cl.R // args.variant_sample)}th) identical to the oracle"}


def _slot_evals(cl) -> int:
    """Sum over live slots of F*S*min(B, q): the (slot, phi, sigma, beta) grid fs_local_config searches."""
    q = cl.states["t"]["q"].astype(np.int64)
    live = np.arange(4)[None, :] < cl.states["n_res"][:, None]
    return int((np.minimum(q, cl.B) * live[:, :, None]).sum()) * cl.F * cl.S


def run_aux_leg(args, torch, dev, workload, flush):
    """configs[3] (`local`) / configs[4] (`consol`): the other two entry points at their own full-size configs.
    Returns the result object (also printed as its own line by --workload local|consol)."""
    import paper_2606_30391_b200 as fs
    import oracle
    cl = synth.make_cluster(workload)
    ctx = fs.Festina(dev.index or 0)
    tb = lambda a: _tb(torch, dev, a)
    ctx.load_profiles(torch.from_numpy(cl.lat).to(dev), torch.from_numpy(cl.pow).to(dev), tb(cl.freq_mhz),
                      tb(cl.models), cl.params)
    d_states = tb(cl.states)
    local = workload == "local"
    rec = 48 if local else 16
    d_out = torch.empty(cl.K * rec, dtype=torch.uint8, device=dev)
    h_states = torch.from_numpy(cl.states.view(np.uint8).reshape(-1).copy()).pin_memory()
    h_out = torch.empty(cl.K * rec, dtype=torch.uint8).pin_memory()
    stream = torch.cuda.current_stream()
    ctx.set_timing(True)
    flags = fs.FS_OBJ_POWER | fs.FS_SPLIT_EXHAUSTIVE      # configs[3]: "minimum-power feasible config"

    def step(states, out, pinned, st):
        ctx.set_gpu_state(states, stream=st, pinned=pinned)
        if local:
            ctx.local_config(flags, n=cl.K, out=out, stream=st, pinned=pinned)
        else:
            ctx.consolidate(out=out, stream=st, pinned=pinned)

    warm = max(args.warmup, 3)
    for _ in range(warm):
        step(d_states, d_out, False, stream)
    torch.cuda.synchronize()
    sampler = ClockSampler(dev.index or 0).start()
    l0 = ctx.launch_count
    kt, dev_ms = {}, 0.0
    for _ in range(args.steps):
        flush.zero_()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(stream); step(d_states, d_out, False, stream); b.record(stream); b.synchronize()
        dev_ms += a.elapsed_time(b)
        for k, v in ctx.get_timing().items():
            kt.setdefault(k, []).append(v)
    launches = ctx.launch_count - l0
    # end to end: the same step on FS_HOST_PINNED buffers (page-locked host memory, the calls enqueue and return,
    # the host waits for the stream before it reads the results), captured once into a CUDA graph
    ctx.set_timing(False)
    for _ in range(3):
        step(h_states, h_out, True, stream)
    torch.cuda.synchronize()
    hgraph = _capture(torch, dev, stream, lambda st: step(h_states, h_out, True, st), f"the {workload} host-buffer step") if args.graph else None
    e2e_t = 0.0
    for _ in range(args.steps):
        flush.zero_(); h_out.zero_(); torch.cuda.synchronize()
        t0 = time.perf_counter()
        if hgraph is not None:
            hgraph.replay()
        else:
            step(h_states, h_out, True, stream)
        torch.cuda.synchronize()
        e2e_t += time.perf_counter() - t0
    clocks = sampler.stop()
    assert np.array_equal(h_out.numpy(), d_out.cpu().numpy()), "host and device paths disagree"
    alu_peak, mhz, peak_src = _alu_peak()
    cores = os.cpu_count() or 1
    if local:
        units, unit_name, metric = _slot_evals(cl), "slot evals/s", "local_slot_evals_per_sec"
        kname, kms, ops, slots = "local_slot_grouped_kernel (a7)", float(np.mean(kt["local_slot"])), 5.0, 5.0
        ops_note = ("5 lane-ops per (slot, phi, sigma, beta) under the power objective: 2 table values, "
                    "rounds*LAT, deadline compare, cost compare/select (6 under the energy objective)")
        res = d_out.cpu().numpy().view(synth.LOCAL_CFG_DT)
        shape = _local_shape(cl, res)
        t0 = time.perf_counter()
        ref = oracle.local_config(cl.lat, cl.pow, cl.states, flags, None, cores)
        dt = time.perf_counter() - t0
        assert np.array_equal(ref["flat"], res["flat"]) and np.array_equal(ref["phi"], res["phi"]) and \
            np.array_equal(ref["beta"], res["beta"]), "CUDA and oracle disagree"
        cpu = {"value": units / dt, "unit": unit_name, "cores": cores, "kind": "oracle",
               "sample": f"the whole config (all {cl.K} GPUs, compared in full), {dt:.1f} s"}
        work = (f"{_workload_name(cl)}: K={cl.K} GPUs, 2-4 co-residents, queue depths U{{0..256}}, "
                f"F={cl.F} x all SM splits (S={cl.S}) x batch 1..{cl.B}; step = fs_set_gpu_state + "
                "fs_local_config(all GPUs, power objective, exhaustive splits)")
        ncu_path = NCU_LOCAL
    else:
        units, unit_name, metric = cl.K * cl.K * cl.F, "pair-frequency evals/s", "consol_pair_freq_evals_per_sec"
        kname, kms, ops, slots = "consol_pair_kernel (a10)", float(np.mean(kt["consol_pair"])), 4.0, 3.25
        ops_note = ("4 lane-ops per (source, destination, phi): int add + compare (feasibility), fp32 add, min; SURVEY "
                    "8(d) lists 8 by counting the two fp32 and two small-int operands as four on-chip loads, which the "
                    "kernel amortises (one broadcast read serves 2 destinations x 32 lanes, one streamed value 8 sources): "
                    "`survey_formula` gives that figure, above 1 for that reason")
        res = d_out.cpu().numpy().view(synth.CONSOL_DT)
        shape = {"has_destination_frac": float((res["dst"] >= 0).mean()),
                 "distinct_destinations": int(len(np.unique(res["dst"][res["dst"] >= 0]))),
                 "hist_phi": _hist(res["phi"][res["dst"] >= 0], cl.F)}
        p = cl.params
        t0 = time.perf_counter()
        ref = oracle.consolidate(cl.lat, cl.pow, cl.models, cl.states, p.p_idle_w, p.horizon_ms, p.mem_cap_mb,
                                 p.delta_pct, cores)
        dt = time.perf_counter() - t0
        assert np.array_equal(ref["dst"], res["dst"]) and np.array_equal(ref["phi"], res["phi"]), "CUDA and oracle disagree"
        cpu = {"value": units / dt, "unit": unit_name, "cores": cores, "kind": "oracle",
               "sample": f"the whole config ({cl.K} sources x {cl.K} destinations, compared in full), {dt:.1f} s"}
        work = (f"{_workload_name(cl)}: K={cl.K} GPUs, M={cl.M}, 1-2 tenants, load ~ Beta(2,5); "
                f"step = fs_set_gpu_state + fs_consolidate ({cl.K * cl.K} pairs x {cl.F} frequencies)")
        ncu_path = NCU_CONSOL
    steps = args.steps
    achieved = ops * units / (kms * 1e-3)
    # instructions the kernel's inner loop issues per unit (local: multiply, compare, predicated min, half a
    # broadcast LDS.128, per-beta set-up shared by 8 rows; consol: 3.25)
    pipe = slots * units / (kms * 1e-3)
    line = {"metric": metric, "value": units * steps / (dev_ms * 1e-3), "unit": unit_name, "n_gpus": 1,
            "steps": steps, "warmup": warm, "ms_per_step": dev_ms / steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": work, "K": cl.K, "M": cl.M, "F": cl.F, "S": cl.S, "B": cl.B,
                       "l2": "flushed between timed steps by overwriting a 256 MiB buffer"},
            "graph": {"device_step": False, "host_step": hgraph is not None},
            "decisions_per_sec": cl.K * steps / (dev_ms * 1e-3),
            "kernel_ms": {k: float(np.mean(v)) for k, v in kt.items()},
            "e2e": {"value": units * steps / e2e_t, "unit": unit_name, "ms_per_step": 1e3 * e2e_t / steps,
                    "h2d_bytes_per_step": cl.K * 128, "d2h_bytes_per_step": cl.K * rec},
            "gpu_launches": int(launches), "clocks": clocks,
            "roofline": {"bound": "alu", "kernel": kname, "achieved": achieved / 1e12, "peak": alu_peak / 1e12,
                         "unit": "Tlane-op/s", "frac": achieved / alu_peak, "traffic": None, "kernel_ms": kms,
                         "peak_pipe": {"instructions_per_unit": slots, "achieved": pipe / 1e12, "frac": pipe / alu_peak,
                                       "note": "instructions the inner loop issues per unit x units / kernel time / the same peak "
                                               "(an issue-slot utilisation from counts, to set beside ncu's issue_active)"},
                         "ncu": _ncu_block(ncu_path),
                         "note": ops_note + f"; x {units} units / CUDA-event time of the kernel; peak = 148 SMs x "
                                 f"128 lanes/clk x sm_max_mhz ({peak_src})"},
            "degeneracy": shape, "cpu_baseline": cpu}
    if not local:
        line["roofline"]["survey_formula"] = {"lane_ops_per_unit": 8.0, "frac": 8.0 * units / (kms * 1e-3) / alu_peak}
    if not line["roofline"]["ncu"].get("missing"):
        line["roofline"]["traffic"] = line["roofline"]["ncu"].get("dram_bytes")
    ctx.close()
    return line


def run_small_leg(args, torch, dev, workload, flush):
    """configs[0] / configs[1]: the pod step at the two small configs (latency-bound: no roofline claim), the
    placements and local configurations compared with the oracle in full."""
    import paper_2606_30391_b200 as fs
    import oracle
    cl = synth.make_cluster(workload)
    ctx = fs.Festina(dev.index or 0)
    tb = lambda a: _tb(torch, dev, a)
    ctx.load_profiles(torch.from_numpy(cl.lat).to(dev), torch.from_numpy(cl.pow).to(dev), tb(cl.freq_mhz),
                      tb(cl.models), cl.params)
    d_states, d_reqs = tb(cl.states), tb(cl.requests)
    d_place = torch.empty(cl.R * 32, dtype=torch.uint8, device=dev)
    d_local = torch.empty(cl.K * 48, dtype=torch.uint8, device=dev)
    stream = torch.cuda.current_stream()

    def step(st):
        ctx.set_gpu_state(d_states, stream=st)
        ctx.place_batch(d_reqs, out=d_place, stream=st)
        ctx.local_config(0, n=cl.K, out=d_local, stream=st)

    for _ in range(3):
        step(stream)
    torch.cuda.synchronize()
    graph = _capture(torch, dev, stream, step, f"the {workload} step") if args.graph else None
    ms = 0.0
    for _ in range(args.steps):
        flush.zero_()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(stream)
        if graph is not None:
            graph.replay()
        else:
            step(stream)
        b.record(stream); b.synchronize()
        ms += a.elapsed_time(b)
    cores = os.cpu_count() or 1
    place = d_place.cpu().numpy().view(synth.PLACEMENT_DT)
    local = d_local.cpu().numpy().view(synth.LOCAL_CFG_DT)
    t0 = time.perf_counter()
    ref = oracle.place_batch(cl.lat, cl.pow, cl.models, cl.states, cl.requests, cores)
    lref = oracle.local_config(cl.lat, cl.pow, cl.states, 0, None, cores)
    dt = time.perf_counter() - t0
    assert np.array_equal(ref["flat"], place["flat"]) and np.array_equal(ref["energy_mj"].view(np.uint32), place["energy_mj"].view(np.uint32))
    assert np.array_equal(lref["flat"], local["flat"]) and np.array_equal(lref["beta"], local["beta"])
    pairs, cand = bench_work.eligible_work(cl)
    shape = _place_shape(cl, place)
    shape.pop("hist_beta")
    ctx.close()
    return {"workload": f"{_workload_name(cl)}: K={cl.K}, M={cl.M}, F={cl.F}, S={cl.S}, B={cl.B}, R={cl.R}",
            "ms_per_step": ms / args.steps, "graph": graph is not None,
            "value": cand * args.steps / (ms * 1e-3), "unit": UNIT,
            "decisions_per_sec": (cl.R + cl.K) * args.steps / (ms * 1e-3), "eligible_candidates_per_step": cand,
            "cpu_baseline": {"value": cand / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
                             "sample": f"the whole config, compared in full, {dt:.2f} s"},
            "degeneracy": shape, "note": "latency-bound at this size: no roofline claim"}


def ncu_import(rep, out_path, command):
    """`ncu -i rep --page raw --csv` -> the small tracked JSON summary the roofline blocks quote (per kernel launch
    in the report; the first one is what bench.py reads).  Runs anywhere ncu is installed: no GPU needed."""
    raw = subprocess.run(["ncu", "-i", rep, "--page", "raw", "--csv"], capture_output=True, text=True, check=True).stdout
    rows = list(csv.reader(raw.splitlines()))
    hdr = rows[0]
    want = {"kernel": "Kernel Name", "duration_ns": "gpu__time_duration.sum",
            "sm_throughput_pct": "sm__throughput.avg.pct_of_peak_sustained_elapsed",
            "issue_active_pct": "smsp__issue_active.avg.pct_of_peak_sustained_active",
            "warp_instructions": "smsp__inst_executed.sum",
            "warps_active_pct": "sm__warps_active.avg.pct_of_peak_sustained_active",
            "dram_read_bytes": "dram__bytes_read.sum", "dram_write_bytes": "dram__bytes_write.sum",
            "pipe_alu_pct": "sm__inst_executed_pipe_alu.avg.pct_of_peak_sustained_active",
            "pipe_fma_pct": "sm__inst_executed_pipe_fma.avg.pct_of_peak_sustained_active",
            "pipe_lsu_pct": "sm__inst_executed_pipe_lsu.avg.pct_of_peak_sustained_active",
            "l1tex_throughput_pct": "l1tex__throughput.avg.pct_of_peak_sustained_elapsed",
            "lts_throughput_pct": "lts__throughput.avg.pct_of_peak_sustained_elapsed",
            "registers_per_thread": "launch__registers_per_thread", "grid": "launch__grid_size", "block": "launch__block_size",
            "sm_clock_ghz": "sm__cycles_elapsed.avg.per_second"}
    units = dict(zip(hdr, rows[1]))
    scale = {"Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "byte": 1.0, "us": 1e3, "ms": 1e6, "ns": 1.0, "s": 1e9}
    launches = []
    for r in rows[2:]:
        d = dict(zip(hdr, r))
        o = {}
        for k, m in want.items():
            if m not in d:
                continue
            v = d[m]
            if k == "kernel":
                o[k] = v.split("(")[0][-120:]
                continue
            try:
                x = float(v.replace(",", ""))
            except ValueError:
                continue
            if k.endswith("_bytes") or k == "duration_ns":
                x *= scale.get(units.get(m, ""), 1.0)
            o[k] = x
        stalls = {k[len("smsp__average_warps_issue_stalled_"):-len("_per_issue_active.ratio")]: float(v)
                  for k, v in d.items() if k.startswith("smsp__average_warps_issue_stalled_") and k.endswith("_per_issue_active.ratio") and v}
        tot = sum(stalls.values()) or 1.0
        o["stall_pct"] = {k: round(100 * v / tot, 1) for k, v in sorted(stalls.items(), key=lambda x: -x[1])[:8]}
        if "dram_read_bytes" in o:
            o["dram_bytes"] = o["dram_read_bytes"] + o.get("dram_write_bytes", 0.0)
        launches.append(o)
    if not launches:
        raise SystemExit(f"no kernel launch in {rep}")
    dirty = bool(subprocess.run(["git", "status", "--porcelain", "--", "paper_2606_30391_b200"], cwd=ROOT, capture_output=True, text=True).stdout.strip())
    summary = dict(launches[0])
    summary.update({"captured_at_git_sha": _git_sha(), "sources_modified_since_that_commit": dirty, "csrc_hash": _csrc_hash(),
                    "command": command, "report": os.path.basename(rep), "launches_in_report": len(launches),
                    "note": "figures of a run under the profiler (cold caches, serialised, ~40 replays): evidence for shares "
                            "and counters, never a bench value"})
    if len(launches) > 1:
        summary["other_launches"] = launches[1:]
    json.dump(summary, open(out_path, "w"), indent=1)
    print(f"wrote {out_path}: {summary.get('kernel')} {summary.get('duration_ns', 0) / 1e3:.1f} us, "
          f"{summary.get('warp_instructions', 0):.0f} warp instructions")


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _spawn_cmd(n, argv):
    """The command line `python bench.py --gpus N` re-executes itself under: one rank per GPU of this node."""
    return [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={n}",
            "--master-addr", "127.0.0.1", "--master-port", str(_free_port()), os.path.abspath(__file__)] + list(argv)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="pod", choices=list(synth.CONFIGS))
    ap.add_argument("--cpu-requests", type=int, default=12288, help="oracle sample of the cpu_baseline leg")
    ap.add_argument("--ref-requests", type=int, default=1024, help="oracle sample per step of --impl reference")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--graph", type=int, default=1, help="1: replay the device step from a CUDA graph")
    ap.add_argument("--split-modes", default="exhaustive", choices=["exhaustive", "both"],
                    help="pod: fs_local_config once (all splits) or twice (all splits, then the per-task minimum-SM rule)")
    ap.add_argument("--overlap", type=int, default=1, help="1: fs_local_config on a second stream beside fs_place_batch")
    ap.add_argument("--variants", type=int, default=1, help="1: time the scoring kernel on the reshaped pod workloads too")
    ap.add_argument("--variant-sample", type=int, default=128, help="requests per variant recomputed by the oracle")
    ap.add_argument("--aux", type=int, default=1, help="1: add the configs[3] / configs[4] / configs[0] / configs[1] legs")
    ap.add_argument("--sustained-s", type=float, default=2.0, help="seconds of back-to-back replays for `sustained` (0: off)")
    ap.add_argument("--detail-out", default=os.path.join(ROOT, "bench_detail.json"),
                    help="where the full result goes (histograms, work counters, notes, ncu summaries); stdout carries the contract line only")
    ap.add_argument("--ncu-import", default=None, help="an .ncu-rep to summarise (with --ncu-out); nothing is run on a GPU")
    ap.add_argument("--ncu-out", default=None)
    ap.add_argument("--ncu-cmd", default="", help="the ncu command line that made the report (recorded in the summary)")
    args = ap.parse_args()
    if args.ncu_import:
        ncu_import(args.ncu_import, args.ncu_out or NCU_POD, args.ncu_cmd)
        return
    if args.impl == "reference":
        run_reference(args)
        return
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        # `python bench.py --gpus N`: start the N ranks here (one process per GPU, NCCL), exactly as the driver's
        # torch.distributed.run command line would
        import torch
        have = torch.cuda.device_count()
        if have < args.gpus:
            raise SystemExit(f"bench.py: --gpus {args.gpus} but only {have} CUDA device(s) are visible")
        os.execv(sys.executable, _spawn_cmd(args.gpus, sys.argv[1:]))
    if args.workload in ("local", "consol"):
        import torch
        ws, rank, lrank = _dist()
        if rank != 0:
            return
        dev = torch.device("cuda", lrank)
        torch.cuda.set_device(dev)
        flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
        emit(run_aux_leg(args, torch, dev, args.workload, flush), args.detail_out)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
