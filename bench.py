#!/usr/bin/env python
"""bench.py — whole-hot-path throughput of libfestina_eval on N B200s (one process per GPU).

A *step* is one pass of the hot path over one batch of synthetic input (BASELINE.json
configs[2], "pod": K=1,024 GPUs, M=64 models, F=64, S=16, B=128, R=65,536 requests):
    fs_set_gpu_state (co-resident summaries)  ->  fs_place_batch (R requests)
    ->  fs_local_config on every GPU.
`value` = nominal dense placement candidates (R*K*S*F) of all ranks / device time of the step,
inputs resident in HBM.  `e2e` = the same through the C ABI with pinned HOST buffers (H2D of
state + requests, D2H of placements + local configs inside the timed region).
N > 1: tables and GPU state are replicated, every rank scores its own R requests (weak scaling,
no data-path collective).
`--impl reference` times the CPU oracle (test infrastructure) on a bounded sample instead.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from paper_2606_30391_b200 import synth  # noqa: E402

METRIC = "placement_candidate_evals_per_sec"
UNIT = "candidates/s"
# DESIGN.md §7 "Roofline": lane-operations (one 32-bit load / arithmetic / compare / select on one
# lane) the method needs per unit of work, for the units the scoring kernel counts itself
OPS_PER_CANDIDATE = 13.0   # dense definition: 8 fp32 arithmetic + 5 compare/select
OPS_TILE = 14.0            # per (request, sigma, phi): 4 table loads, 5 fp32, 2 tests, 3 running minima
OPS_PAIR_TEST = 18.0       # per (request, GPU) tested: 8-word record, 7 eligibility compares, bound (2 fp32 + compare)
OPS_TSTAR = 12.0           # per swept pair: deadline threshold T*
OPS_SWEEP = 2.0            # per swept candidate: compare + predicated min
OPS_ROW = 4.0              # per swept (pair, phi): A0 load, add, min, subtract/compare share
OPS_WARM_TEST = 20.0       # per warm pair tested: 12-word item, bound (5 fp32), 3 compares
OPS_DEF = 14.0             # per candidate scored by the definition: 4 loads, 4 mul, 3 add/sub, 3 compares
# dram bytes per launch of the scoring kernel and its issue utilisation, from the committed ncu
# capture of this workload (profiles/; a profiler cannot run inside the timed bench)
NCU_TRAFFIC_BYTES = 42.45e6
NCU_NOTE = {"source": "profiles/r01_final_pod.md (ncu --set full of this kernel on this workload)",
            "sm_throughput_pct_of_peak": 65.1, "issue_active_pct_of_peak": 70.4, "warp_instructions": 199.8e6,
            "note": "executed instructions; `frac` above counts only the lane-operations the method needs"}
SM_COUNT, ISSUE_LANES_PER_CLK_PER_SM = 148, 128   # 4 schedulers x 32 lanes (B300_MICROARCH "issue")


def _peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return json.load(open(p)), "measured"
        except Exception:
            pass
    return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0}, "fallback"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.rows, self.proc, self.thr = [], None, None
        self.cmd = ["nvidia-smi", f"--id={index}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                    "-lms", "100"]

    def start(self):
        try:
            self.proc = subprocess.Popen(self.cmd, stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except OSError:
            return
        def pump():
            for line in self.proc.stdout:
                self.rows.append([x.strip() for x in line.split(",")])
        self.thr = threading.Thread(target=pump, daemon=True)
        self.thr.start()

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


def oracle_sample(cl, n_req: int, nthreads: int):
    """One bounded pass of the hot path through the CPU oracle; returns (seconds, candidates)."""
    import oracle
    n_gpu = max(1, int(round(cl.K * n_req / cl.R)))
    t0 = time.perf_counter()
    oracle.place_batch(cl.lat, cl.pow, cl.models, cl.states, cl.requests[:n_req], nthreads)
    oracle.local_config(cl.lat, cl.pow, cl.states, 0, np.arange(n_gpu, dtype=np.int32), nthreads)
    dt = time.perf_counter() - t0
    return dt, n_req * cl.K * cl.S * cl.F, n_gpu


def run_reference(args):
    ws, rank, _ = _dist()
    if rank != 0:
        return
    cl = synth.make_cluster(args.workload)
    cores = os.cpu_count() or 1
    n_req = args.ref_requests
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
            "data": "synthetic", "config": _config(cl, args),
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def _config(cl, args):
    return {"workload": f"{cl.name} (BASELINE.json configs[2]): K={cl.K} GPUs, M={cl.M}, F={cl.F}, S={cl.S}, "
                        f"B={cl.B}, R={cl.R} requests per rank; step = fs_set_gpu_state + fs_place_batch + "
                        f"fs_local_config(all GPUs, energy objective, exhaustive splits" + (", then the minimum-SM split rule" if args.split_modes == "both" else "") + ")" + ("; the two calls on two streams" if args.overlap else "") + ("; one CUDA graph per step" if args.graph else ""),
            "K": cl.K, "M": cl.M, "F": cl.F, "S": cl.S, "B": cl.B, "R_per_rank": cl.R,
            "l2": "flushed between timed steps by overwriting a 256 MiB buffer",
            "parallelism": f"replicated tables+state, requests sharded x{args.gpus}"}


def run_ours(args):
    import torch
    import paper_2606_30391_b200 as fs

    ws, rank, lrank = _dist()
    dist = None
    if ws > 1:
        import torch.distributed as dist
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        torch.cuda.set_device(lrank)
        dist.init_process_group("nccl", device_id=torch.device("cuda", lrank))
    dev = torch.device("cuda", lrank)
    torch.cuda.set_device(dev)
    cl = synth.make_cluster(args.workload)
    if rank > 0:   # every rank scores its own batch
        cl.requests = synth.make_requests(cl.seed + 7919 * rank, cl.R, cl.M)
    ctx = fs.Festina(lrank)
    tb = lambda a: torch.from_numpy(np.ascontiguousarray(a).view(np.uint8).reshape(-1)).to(dev)
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

    def step_device(serial=False, st=None):
        st = stream if st is None else st
        ctx.set_gpu_state(d_states, stream=st)
        if side is None or serial:
            ctx.place_batch(d_reqs, out=d_place, stream=st)
            ctx.local_config(0, n=cl.K, out=d_local, stream=st)
            if both_splits:
                ctx.local_config(2, n=cl.K, out=d_local2, stream=st)
            return
        ev_state.record(st)
        side.wait_event(ev_state)
        ctx.local_config(0, n=cl.K, out=d_local, stream=side)
        if both_splits:
            ctx.local_config(2, n=cl.K, out=d_local2, stream=side)
        ctx.place_batch(d_reqs, out=d_place, stream=st)
        ev_side.record(side)
        st.wait_event(ev_side)

    def barrier():
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
            torch.cuda.synchronize()

    for _ in range(max(args.warmup, 3)):
        step_device()
    barrier()
    # The calls are asynchronous and allocation-free after the first step, so a whole step (fork to the second
    # stream and join included) can be captured into a CUDA graph and replayed: one launch per step for the host.
    graph, launches_per_step = None, None
    if args.graph:
        try:
            ctx.set_timing(False)                       # event records of the per-kernel timers are not capturable
            cap = torch.cuda.Stream(device=dev)
            cap.wait_stream(stream)
            lc = ctx.launch_count
            graph = torch.cuda.CUDAGraph()
            with torch.cuda.graph(graph, stream=cap):
                step_device(st=torch.cuda.current_stream())
            launches_per_step = ctx.launch_count - lc
            stream.wait_stream(cap)
            for _ in range(3):
                graph.replay()
            torch.cuda.synchronize()
        except Exception as e:                          # noqa: BLE001 - fall back to direct launches
            print(f"bench.py: CUDA graph capture failed ({e}); timing direct launches", file=sys.stderr)
            graph = None
        ctx.set_timing(True)
    barrier()
    sampler = ClockSampler(lrank)
    sampler.start()
    l0 = ctx.launch_count
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
    launches = ctx.launch_count - l0 if graph is None else launches_per_step * args.steps
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
    # work counters: one untimed call of the counting instantiation (same input, same work)
    ctx.set_work_stats(True)
    ctx.place_batch(d_reqs, out=d_place, stream=stream)
    pstats = ctx.last_place_stats()
    ctx.set_work_stats(False)
    useful_ops = (OPS_TILE * pstats["requests"] * cl.S * cl.F + OPS_PAIR_TEST * 32 * pstats["chunks_tested"]
                  + OPS_TSTAR * pstats["cold_pairs_swept"] + OPS_SWEEP * pstats["cold_candidates_swept"]
                  + OPS_ROW * cl.F * pstats["cold_pairs_swept"] + OPS_WARM_TEST * pstats["warm_pairs_tested"]
                  + OPS_DEF * pstats["candidates_scored"])
    # the dense definition's work: every eligible (request, GPU) pair x sm_free x F, counted by the
    # generic kernel (no pruning) on a second context; also an on-GPU cross-check of the two kernels
    os.environ["FS_FORCE_GENERIC"] = "1"
    ctx_g = fs.Festina(lrank)
    del os.environ["FS_FORCE_GENERIC"]
    ctx_g.load_profiles(torch.from_numpy(cl.lat).to(dev), torch.from_numpy(cl.pow).to(dev), tb(cl.freq_mhz),
                        tb(cl.models), cl.params)
    ctx_g.set_gpu_state(d_states, stream=stream)
    ctx_g.set_work_stats(True)
    d_place_g = torch.empty_like(d_place)
    ctx_g.place_batch(d_reqs, out=d_place_g, stream=stream)
    gstats = ctx_g.last_place_stats()
    torch.cuda.synchronize()
    assert torch.equal(d_place_g, d_place), "generic and dense scoring kernels disagree"
    ctx_g.close()
    pairs, cand_def = gstats["cold_pairs_eligible"], gstats["candidates_scored"]

    # end to end through the C ABI with pinned host buffers
    h_states = torch.from_numpy(cl.states.view(np.uint8).reshape(-1).copy()).pin_memory()
    h_reqs = torch.from_numpy(cl.requests.view(np.uint8).reshape(-1).copy()).pin_memory()
    h_place = torch.empty(cl.R * 32, dtype=torch.uint8).pin_memory()
    h_local = torch.empty(cl.K * 48, dtype=torch.uint8).pin_memory()
    h_local2 = torch.empty(cl.K * 48, dtype=torch.uint8).pin_memory()

    # The same step as above with FS_HOST_PINNED buffers: every step copies its inputs (state records, requests)
    # from page-locked host memory and its results (placements, local configurations) back; the host waits for
    # the stream before it reads them.  Two streams and one CUDA graph per step, as in the device-resident step.
    def step_host(st=None):
        st = stream if st is None else st
        ctx.set_gpu_state(h_states, stream=st, pinned=True)
        if side is None:
            ctx.place_batch(h_reqs, out=h_place, stream=st, pinned=True)
            ctx.local_config(0, n=cl.K, out=h_local, stream=st, pinned=True)
            if both_splits:
                ctx.local_config(2, n=cl.K, out=h_local2, stream=st, pinned=True)
            return
        ev_state.record(st)
        side.wait_event(ev_state)
        ctx.local_config(0, n=cl.K, out=h_local, stream=side, pinned=True)
        if both_splits:
            ctx.local_config(2, n=cl.K, out=h_local2, stream=side, pinned=True)
        ctx.place_batch(h_reqs, out=h_place, stream=st, pinned=True)
        ev_side.record(side)
        st.wait_event(ev_side)

    ctx.set_timing(False)
    for _ in range(3):
        step_host()
    torch.cuda.synchronize()
    hgraph = None
    if args.graph:
        try:
            cap = torch.cuda.Stream(device=dev)
            cap.wait_stream(stream)
            hgraph = torch.cuda.CUDAGraph()
            with torch.cuda.graph(hgraph, stream=cap):
                step_host(st=torch.cuda.current_stream())
            stream.wait_stream(cap)
            for _ in range(3):
                hgraph.replay()
            torch.cuda.synchronize()
        except Exception as e:                          # noqa: BLE001 - fall back to direct calls
            print(f"bench.py: CUDA graph capture of the host-buffer step failed ({e}); timing direct calls", file=sys.stderr)
            hgraph = None
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

    t = torch.tensor([dev_ms, e2e_t * 1e3, wall * 1e3], dtype=torch.float64, device=dev)
    if dist is not None:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dev_ms, e2e_ms, wall_ms = (float(x) for x in t.cpu())
    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return
    grid_cands = cl.R * cl.K * cl.S * cl.F
    steps = args.steps
    value = ws * grid_cands * steps / (dev_ms * 1e-3)
    peaks, peak_src = _peaks()
    sm_clk_hz = float(peaks.get("sm_max_mhz", 1965.0)) * 1e6
    alu_peak = SM_COUNT * ISSUE_LANES_PER_CLK_PER_SM * sm_clk_hz          # lane-instructions / s
    score_ms = float(np.mean(kt.get("place_score", [float("nan")])))
    achieved = useful_ops / (score_ms * 1e-3)
    nominal = OPS_PER_CANDIDATE * cand_def / (score_ms * 1e-3)
    place = d_place.cpu().numpy().view(synth.PLACEMENT_DT)
    ok = place["gpu"] >= 0
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": ws, "steps": steps, "warmup": max(args.warmup, 3),
        "ms_per_step": dev_ms / steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32", "data": "synthetic", "config": _config(cl, args),
        "decisions_per_sec": ws * (cl.R + cl.K) * steps / (dev_ms * 1e-3),
        "placement_decisions_per_sec": ws * cl.R * steps / (dev_ms * 1e-3),
        "nominal_candidates_per_step": grid_cands, "eligible_candidates_per_step": cand_def,
        "eligible_pairs_per_step": pairs, "place_stats": pstats,
        "kernel_ms": {k: float(np.mean(v)) for k, v in kt.items()},
        "serial": {"ms_per_step": serial_ms / steps,
                   "note": ("timed steps run fs_place_batch and fs_local_config on two streams"
                            + (", replayed from one CUDA graph per step" if graph is not None else "")
                            + "; kernel_ms and the roofline come from the same steps run serially, launch by launch, "
                              "right after" if (args.overlap or graph is not None) else
                            "timed steps are serial: kernel_ms comes from them")},
        "wall_ms_per_step_incl_flush": wall_ms / steps,
        "e2e": {"value": ws * grid_cands * steps / (e2e_ms * 1e-3), "unit": UNIT, "ms_per_step": e2e_ms / steps,
                "h2d_bytes_per_step": cl.K * 128 + cl.R * 32, "d2h_bytes_per_step": cl.R * 32 + cl.K * 48 * (2 if both_splits else 1),
                "mode": "FS_HOST_PINNED buffers (page-locked host memory): state records and local configurations by "
                        "copy engine, requests read and placement records written over PCIe by the scoring kernel itself"
                        + (", two streams" if side is not None else "") + (", one CUDA graph per step" if hgraph is not None else "")
                        + "; host wall clock around the step incl. the final stream synchronisation"},
        "gpu_launches": int(launches),
        "clocks": clocks,
        "roofline": {"bound": "alu", "kernel": "place_dense_kernel (fs_place_batch scoring + argmin)",
                     "achieved": achieved / 1e12, "peak": alu_peak / 1e12, "unit": "Tlane-op/s",
                     "frac": achieved / alu_peak, "traffic": NCU_TRAFFIC_BYTES,
                     "useful_lane_ops_per_launch": useful_ops, "kernel_ms": score_ms,
                     "dense_definition": {"achieved": nominal / 1e12, "frac": nominal / alu_peak,
                                          "note": f"{OPS_PER_CANDIDATE:g} lane-ops x {cand_def} eligible candidates "
                                                  "(counted by the unpruned generic kernel); above 1 because "
                                                  "exact pruning skips most of them"},
                     "ncu": NCU_NOTE,
                     "note": "achieved = lane-ops of the units the kernel counted itself (DESIGN.md section 7 "
                             "per-unit figures) / CUDA-event time of the launch; peak = 148 SMs x 128 lanes/clk x "
                             f"{sm_clk_hz / 1e6:.0f} MHz ({peak_src} sm_max_mhz); traffic from the committed ncu capture"},
        "degeneracy": {"placed_frac": float(ok.mean()),
                       "top_phi_share": float(np.bincount(place["phi"][ok]).max() / max(ok.sum(), 1)),
                       "distinct_gpus": int(len(np.unique(place["gpu"][ok])))},
    }
    if ws == 1 and not args.no_cpu_baseline:
        cores = os.cpu_count() or 1
        dt, c, n_gpu = oracle_sample(cl, args.cpu_requests, cores)
        line["cpu_baseline"] = {"value": c / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
                                "sample": f"{args.cpu_requests} of {cl.R} requests x all {cl.K} GPUs + "
                                          f"{n_gpu} GPUs local config, {dt:.1f} s"}
    print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()


def _slot_evals(cl) -> int:
    """Sum over live slots of F*S*min(B, q): the (slot, phi, sigma, beta) grid fs_local_config searches."""
    q = cl.states["t"]["q"].astype(np.int64)
    live = np.arange(4)[None, :] < cl.states["n_res"][:, None]
    return int((np.minimum(q, cl.B) * live[:, :, None]).sum()) * cl.F * cl.S


def run_aux(args):
    """--workload local (BASELINE.json configs[3]) / consol (configs[4]): the other two entry points at
    their own full-size configs, same JSON contract.  1 GPU."""
    import torch
    import paper_2606_30391_b200 as fs
    import oracle
    ws, rank, lrank = _dist()
    assert ws == 1, "the local / consol workloads are single-GPU bench lines"
    dev = torch.device("cuda", lrank)
    torch.cuda.set_device(dev)
    cl = synth.make_cluster(args.workload)
    ctx = fs.Festina(lrank)
    tb = lambda a: torch.from_numpy(np.ascontiguousarray(a).view(np.uint8).reshape(-1)).to(dev)
    ctx.load_profiles(torch.from_numpy(cl.lat).to(dev), torch.from_numpy(cl.pow).to(dev), tb(cl.freq_mhz),
                      tb(cl.models), cl.params)
    d_states = tb(cl.states)
    local = args.workload == "local"
    rec = 48 if local else 16
    d_out = torch.empty(cl.K * rec, dtype=torch.uint8, device=dev)
    h_states = torch.from_numpy(cl.states.view(np.uint8).reshape(-1).copy()).pin_memory()
    h_out = torch.empty(cl.K * rec, dtype=torch.uint8).pin_memory()
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    stream = torch.cuda.current_stream()
    ctx.set_timing(True)
    flags = fs.FS_OBJ_POWER | fs.FS_SPLIT_EXHAUSTIVE      # configs[3]: "minimum-power feasible config"

    def step(states, out):
        ctx.set_gpu_state(states, stream=stream)
        if local:
            ctx.local_config(flags, n=cl.K, out=out, stream=stream)
        else:
            ctx.consolidate(out=out, stream=stream)

    warm = max(args.warmup, 3)
    for _ in range(warm):
        step(d_states, d_out)
    torch.cuda.synchronize()
    sampler = ClockSampler(lrank)
    sampler.start()
    l0 = ctx.launch_count
    kt, dev_ms = {}, 0.0
    for _ in range(args.steps):
        flush.zero_()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(stream); step(d_states, d_out); b.record(stream); b.synchronize()
        dev_ms += a.elapsed_time(b)
        for k, v in ctx.get_timing().items():
            kt.setdefault(k, []).append(v)
    launches = ctx.launch_count - l0
    # end to end: the same step on FS_HOST_PINNED buffers (page-locked host memory, the calls enqueue and return,
    # the host waits for the stream before it reads the results), captured once into a CUDA graph
    ctx.set_timing(False)

    def step_host():
        ctx.set_gpu_state(h_states, stream=torch.cuda.current_stream(), pinned=True)
        if local:
            ctx.local_config(flags, n=cl.K, out=h_out, stream=torch.cuda.current_stream(), pinned=True)
        else:
            ctx.consolidate(out=h_out, stream=torch.cuda.current_stream(), pinned=True)

    for _ in range(3):
        step_host()
    torch.cuda.synchronize()
    hgraph = None
    if args.graph:
        try:
            cap = torch.cuda.Stream(device=dev)
            cap.wait_stream(stream)
            hgraph = torch.cuda.CUDAGraph()
            with torch.cuda.graph(hgraph, stream=cap):
                step_host()
            stream.wait_stream(cap)
            for _ in range(3):
                hgraph.replay()
            torch.cuda.synchronize()
        except Exception as e:                          # noqa: BLE001 - fall back to direct calls
            print(f"bench.py: CUDA graph capture of the host-buffer step failed ({e}); timing direct calls", file=sys.stderr)
            hgraph = None
    e2e_t = 0.0
    for _ in range(args.steps):
        flush.zero_(); h_out.zero_(); torch.cuda.synchronize()
        t0 = time.perf_counter()
        if hgraph is not None:
            hgraph.replay()
        else:
            step_host()
        torch.cuda.synchronize()
        e2e_t += time.perf_counter() - t0
    assert np.array_equal(h_out.numpy(), d_out.cpu().numpy()), "host and device paths disagree"
    clocks = sampler.stop()
    assert np.array_equal(h_out.numpy(), d_out.cpu().numpy()), "host and device paths disagree"
    peaks, peak_src = _peaks()
    alu_peak = SM_COUNT * ISSUE_LANES_PER_CLK_PER_SM * float(peaks.get("sm_max_mhz", 1965.0)) * 1e6
    cores = os.cpu_count() or 1
    if local:
        units, unit_name, metric = _slot_evals(cl), "slot evals/s", "local_slot_evals_per_sec"
        kname, kms, ops = "local_slot_grouped_kernel (a7)", float(np.mean(kt["local_slot"])), 5.0
        ops_note = ("5 lane-ops per (slot, phi, sigma, beta) under the power objective: 2 table values, "
                    "rounds*LAT, deadline compare, cost compare/select (6 under the energy objective)")
        res = d_out.cpu().numpy().view(synth.LOCAL_CFG_DT)
        degeneracy = {"feasible_frac": float((res["phi"] >= 0).mean()),
                      "top_phi_share": float(np.bincount(res["phi"][res["phi"] >= 0]).max() / max((res["phi"] >= 0).sum(), 1))}
        n_s = args.cpu_gpus
        t0 = time.perf_counter()
        ref = oracle.local_config(cl.lat, cl.pow, cl.states, flags, np.arange(n_s, dtype=np.int32), cores)
        dt = time.perf_counter() - t0
        assert np.array_equal(ref["flat"], res["flat"][:n_s]), "CUDA and oracle disagree on the sample"
        sub = synth.Cluster(**{**cl.__dict__, "states": cl.states[:n_s], "K": n_s})
        cpu = {"value": _slot_evals(sub) / dt, "unit": unit_name, "cores": cores, "kind": "oracle",
               "sample": f"GPUs 0..{n_s - 1} of {cl.K}, {dt:.1f} s"}
        work = (f"local (BASELINE.json configs[3]): K={cl.K} GPUs, 2-4 co-residents, queue depths U{{0..256}}, "
                f"F={cl.F} x all SM splits (S={cl.S}) x batch 1..{cl.B}; step = fs_set_gpu_state + "
                "fs_local_config(all GPUs, power objective, exhaustive splits)")
        decisions = cl.K
    else:
        units, unit_name, metric = cl.K * cl.K * cl.F, "pair-frequency evals/s", "consol_pair_freq_evals_per_sec"
        kname, kms, ops = "consol_pair_kernel (a10)", float(np.mean(kt["consol_pair"])), 8.0
        ops_note = ("8 lane-ops per (source, destination, phi): 2 fp32 + 2 small-int values, int add + compare, "
                    "fp32 add, min (SURVEY 8(d))")
        res = d_out.cpu().numpy().view(synth.CONSOL_DT)
        degeneracy = {"has_destination_frac": float((res["dst"] >= 0).mean()),
                      "distinct_destinations": int(len(np.unique(res["dst"][res["dst"] >= 0])))}
        p = cl.params
        t0 = time.perf_counter()
        ref = oracle.consolidate(cl.lat, cl.pow, cl.models, cl.states, p.p_idle_w, p.horizon_ms, p.mem_cap_mb,
                                 p.delta_pct, cores)
        dt = time.perf_counter() - t0
        assert np.array_equal(ref["dst"], res["dst"]), "CUDA and oracle disagree"
        cpu = {"value": units / dt, "unit": unit_name, "cores": cores, "kind": "oracle",
               "sample": f"the whole config ({cl.K} sources x {cl.K} destinations), {dt:.1f} s"}
        work = (f"consol (BASELINE.json configs[4]): K={cl.K} GPUs, M={cl.M}, 1-2 tenants, load ~ Beta(2,5); "
                f"step = fs_set_gpu_state + fs_consolidate ({cl.K * cl.K} pairs x {cl.F} frequencies)")
        decisions = cl.K
    steps = args.steps
    achieved = ops * units / (kms * 1e-3)
    line = {"metric": metric, "value": units * steps / (dev_ms * 1e-3), "unit": unit_name, "n_gpus": 1,
            "steps": steps, "warmup": warm, "ms_per_step": dev_ms / steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": work, "K": cl.K, "M": cl.M, "F": cl.F, "S": cl.S, "B": cl.B,
                       "l2": "flushed between timed steps by overwriting a 256 MiB buffer"},
            "decisions_per_sec": decisions * steps / (dev_ms * 1e-3),
            "kernel_ms": {k: float(np.mean(v)) for k, v in kt.items()},
            "e2e": {"value": units * steps / e2e_t, "unit": unit_name, "ms_per_step": 1e3 * e2e_t / steps,
                    "h2d_bytes_per_step": cl.K * 128, "d2h_bytes_per_step": cl.K * rec},
            "gpu_launches": int(launches), "clocks": clocks,
            "roofline": {"bound": "alu", "kernel": kname, "achieved": achieved / 1e12, "peak": alu_peak / 1e12,
                         "unit": "Tlane-op/s", "frac": achieved / alu_peak, "traffic": None, "kernel_ms": kms,
                         "note": ops_note + f"; x {units} units / CUDA-event time of the kernel; peak = 148 SMs x "
                                 f"128 lanes/clk x sm_max_mhz ({peak_src})"},
            "degeneracy": degeneracy, "cpu_baseline": cpu}
    print(json.dumps(line), flush=True)
    ctx.close()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="pod", choices=list(synth.CONFIGS))
    ap.add_argument("--cpu-requests", type=int, default=12288, help="oracle sample of the cpu_baseline leg")
    ap.add_argument("--ref-requests", type=int, default=1024, help="oracle sample per step of --impl reference")
    ap.add_argument("--cpu-gpus", type=int, default=4096, help="oracle sample (GPUs) of --workload local")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--graph", type=int, default=1, help="1: replay the device step from a CUDA graph")
    ap.add_argument("--split-modes", default="exhaustive", choices=["exhaustive", "both"],
                    help="pod: fs_local_config once (all splits) or twice (all splits, then the per-task minimum-SM rule)")
    ap.add_argument("--overlap", type=int, default=1, help="1: fs_local_config on a second stream beside fs_place_batch")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    elif args.workload in ("local", "consol"):
        run_aux(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
