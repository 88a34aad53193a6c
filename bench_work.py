"""bench_work.py — what bench.py and the tests need around the synthetic clusters that is NOT input generation:
the reshaped variants of a config on which the placement kernel's pruning has less (or nothing) to hold on to, and
the size of the dense definition's candidate set (the denominator-free unit of bench.py's rates).  `eligible_work`
restates the method's eligibility rule (5 % pad, Req_mem, free shares, cold-slot cap, bucket < B), which is why it
lives here beside bench.py and not in the product package: paper_2606_30391_b200/synth.py holds record layouts and
seeded draws only.  Checked against a double loop in tests/test_synth_counts.py."""
from __future__ import annotations

import numpy as np

from paper_2606_30391_b200.synth import Cluster, Stream, make_cluster

# ---- variants of a config on which the placement kernel's pruning has less (or nothing) to hold on to ------
VARIANTS = ("dynamic_power_x4", "cold_starts_feasible", "ties", "identical_gpus")


def make_variant(name: str, variant: str) -> Cluster:
    """configs[name] reshaped (bench.py --variants, tests):
    dynamic_power_x4      4x the dynamic power (everything above a table's lowest-frequency entry): the chosen
                          frequencies spread over the levels instead of piling up at F-1;
    cold_starts_feasible  weight loads 20x cheaper: cold starts meet the TTFT deadline, the sorted cold scan works;
    ties                  tables quantised to a few powers of two and every SLO relaxed: exact ties across GPUs,
                          shares and frequencies, so no lower bound is strict and every eligible pair is swept
                          (ties inside a GPU; the GPUs still differ, so the scan over GPUs still stops early);
    identical_gpus        the adversarial case for branch and bound: eight GPU records repeated K/8 times, hosting
                          only models no request asks for (every pair is a cold start), TTFT deadlines 4x longer
                          (cold starts feasible): the GPUs of the best kind tie EXACTLY, no lower bound separates
                          them and every one of them is swept for every request."""
    cl = make_cluster(name)
    if variant == "dynamic_power_x4":
        cl.pow = (cl.pow + 3.0 * (cl.pow - cl.pow[:, :, :1])).astype(np.float32)
    elif variant == "cold_starts_feasible":
        cl.models["load_ms"] *= 0.05
    elif variant == "ties":
        st = Stream(cl.seed, "ties")
        n = cl.lat.size
        cl.lat[...] = (2.0 ** st.randint(n, 0, 2)).reshape(cl.lat.shape).astype(np.float32)
        cl.pow[...] = (64.0 * 2.0 ** st.randint(n, 0, 1)).reshape(cl.pow.shape).astype(np.float32)
        cl.requests["slo_ttft_ms"] = 1e9
        cl.requests["slo_tbt_ms"] = 1e9
        cl.states["t"]["slo_ms"][...] = 1e9
    elif variant == "identical_gpus":
        half = max(cl.M // 2, 1)
        cl.states[...] = cl.states[np.arange(cl.K) % 8]
        cl.states["t"]["model"][...] = (cl.states["t"]["model"] % half + (cl.M - half)).astype(cl.states["t"]["model"].dtype)
        cl.requests["model"] = cl.requests["model"] % max(cl.M - half, 1)
        cl.requests["slo_ttft_ms"] *= 4.0
    else:
        raise ValueError(f"unknown variant {variant!r}")
    cl.name = f"{name}/{variant}"
    return cl


def eligible_work(cl: Cluster, reqs: np.ndarray | None = None):
    """(eligible (request, GPU) pairs, candidates = sum over them of sm_free * F): the size of the dense
    definition's candidate set (what a scorer without pruning evaluates).  Index bookkeeping for bench.py's
    rates; the one product is the request's memory demand, rounded as the records are (binary32)."""
    reqs = cl.requests if reqs is None else reqs
    st = cl.states
    n_res = st["n_res"].astype(np.int64)
    live = np.arange(4)[None, :] < n_res[:, None]
    smf = cl.S - ((st["t"]["sigma"].astype(np.int64) + 1) * live).sum(axis=1)
    mem_free = st["mem_free_mb"].astype(np.float32)
    O = (21 * reqs["o_pred"].astype(np.int64) + 19) // 20
    mem = (reqs["L"].astype(np.int64) + O).astype(np.float32) * cl.models["kv_mb_per_token"][reqs["model"]].astype(np.float32)
    pairs = cands = 0
    for m in range(cl.M):
        rm = np.sort(mem[reqs["model"] == m])
        if rm.size == 0:
            continue
        hosts = (st["t"]["model"] == m) & live
        warm = hosts.any(axis=1)
        j = np.argmax(hosts, axis=1)                                    # lowest slot holding the model
        kk = np.arange(cl.K)
        q1 = st["t"]["q"][kk, j, 1]
        br1 = np.where(q1 > 0, st["t"]["beta"][kk, j, 1].astype(np.int64) + 1, 0)
        ok = (n_res >= 1) & (smf >= 1) & np.where(warm, br1 < cl.B, n_res < 4)
        # a GPU counts for the requests whose demand is <= its free memory
        cnt = np.searchsorted(rm, mem_free[ok], side="right").astype(np.int64)
        pairs += int(cnt.sum())
        cands += int((cnt * smf[ok]).sum()) * cl.F
    return pairs, cands
