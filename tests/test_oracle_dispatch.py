"""Pins of the oracle's paper-mode dispatcher (Phase 1 feasibility at
F_curr / SM_free, Phase 2 Eq. 2-3 energy argmin with the 2 % stability tie-breaker, Phase 3
F_max retry in T_avail order and scale-out).  CPU only."""
from __future__ import annotations

import numpy as np
import pytest

import oracle
from fs_brute import _slot, f32, INF
from paper_2606_30391_b200 import synth


def _gpu(st, k, model, sigma_used, f_cur, t_avail, mem_free, q1=0, beta1=0):
    """One tenant `model` holding sigma_used share units, queues empty unless q1 is given."""
    st["n_res"][k] = 1; st["f_cur"][k] = f_cur; st["t_avail_ms"][k] = t_avail; st["mem_free_mb"][k] = mem_free
    t = st["t"][k][0]
    t["model"] = model; t["sigma"] = sigma_used - 1; t["beta"] = (0, beta1); t["q"] = (0, q1)
    t["slo_ms"] = (1e9, 1e9)
    st["t"][k][0] = t


def _restate(cl, r):
    """Independent restatement of the three phases for request r: returns (gpu, sigma, phi, phase, E)."""
    rq = cl.requests[r]; m = int(rq["model"]); L = int(rq["L"])
    O = (21 * int(rq["o_pred"]) + 19) // 20
    mem = f32(f32(L + O) * cl.models["kv_mb_per_token"][m])
    rows = []                                             # eligible GPUs: (k, smf, br1, wait)
    for k in range(cl.K):
        g = cl.states[k]; n = int(g["n_res"])
        if n < 1 or not (mem <= g["mem_free_mb"]):
            continue
        smf = cl.S - sum(int(g["t"][i]["sigma"]) + 1 for i in range(n))
        js = [i for i in range(n) if int(g["t"][i]["model"]) == m]
        j = js[0] if js else -1
        br1 = int(g["t"][j]["beta"][1]) + 1 if (j >= 0 and g["t"][j]["q"][1] > 0) else 0
        if smf < 1 or (j < 0 and n >= 4) or br1 >= cl.B:
            continue
        wait = g["t_avail_ms"] if j >= 0 else f32(g["t_avail_ms"] + cl.models["load_ms"][m])
        rows.append((k, smf, br1, wait))

    def own(phi, sg, br1, wait):
        ok0, t0, e0 = _slot(cl.lat, cl.pow, m, 0, phi, sg, max(min(L, cl.B) - 1, 0), L, wait, rq["slo_ttft_ms"])
        ok1, _, e1 = _slot(cl.lat, cl.pow, m, 1, phi, sg, br1, O, 0.0, rq["slo_tbt_ms"])
        e = f32(e0 + e1)
        return (ok0 and ok1 and e < INF), e

    cur = [(k, smf, own(int(cl.states["f_cur"][k]), smf - 1, br1, wait)) for k, smf, br1, wait in rows]
    feas = [(k, smf, e) for k, smf, (ok, e) in cur if ok]
    if feas:
        band = f32(f32(1.02) * min(e for _, _, e in feas))
        near = [(-float(cl.states["mem_free_mb"][k]), -smf, k, e) for k, smf, e in feas if e <= band]
        _, nsmf, k, e = min(near)
        return k, -nsmf - 1, int(cl.states["f_cur"][k]), 1, e
    fmax = [(float(cl.states["t_avail_ms"][k]), k, smf, own(cl.F - 1, smf - 1, br1, wait)) for k, smf, br1, wait in rows]
    fmax = [(ta, k, smf, oe[1]) for ta, k, smf, oe in fmax if oe[0]]
    if fmax:
        _, k, smf, e = min(fmax)
        return k, smf - 1, cl.F - 1, 2, e
    fresh = [(own(phi, cl.S - 1, 0, cl.models["load_ms"][m]), phi) for phi in range(cl.F)]
    fresh = [(float(e), phi, e) for (ok, e), phi in fresh if ok]
    if fresh:
        _, phi, e = min(fresh)
        return -1, cl.S - 1, phi, 3, e
    return -1, -1, -1, -1, INF


@pytest.mark.parametrize("seed", range(30))
def test_dispatch_equals_independent_restatement(seed):
    cl = synth.make_custom(seed=900 + seed, K=[3, 6, 11][seed % 3], M=3, F=5, S=[4, 8][seed % 2], B=6, R=24, lo=1, hi=4)
    if seed % 4 == 1:
        cl.requests["slo_ttft_ms"] *= 0.02             # drives requests into phases 2 and 3
    if seed % 4 == 2:
        cl.states["mem_free_mb"] = 1.0                 # nothing fits anywhere: scale-out for all
    if seed % 4 == 3:
        cl.requests["slo_tbt_ms"] = 1e-3               # not even a fresh GPU helps
    got = oracle.dispatch(cl.lat, cl.pow, cl.models, cl.states, cl.requests)
    for r in range(cl.R):
        k, sg, phi, phase, e = _restate(cl, r)
        o = got[r]
        assert (int(o["gpu"]), int(o["sigma"]), int(o["phi"]), int(o["f_req"])) == (k, sg, phi, phase), (seed, r)
        assert o["energy_mj"] == e or (np.isinf(o["energy_mj"]) and np.isinf(e))


def test_restatement_cases_cover_all_phases():
    seen = set()
    for seed in range(30):
        cl = synth.make_custom(seed=900 + seed, K=[3, 6, 11][seed % 3], M=3, F=5, S=[4, 8][seed % 2], B=6, R=24, lo=1, hi=4)
        if seed % 4 == 1:
            cl.requests["slo_ttft_ms"] *= 0.02
        if seed % 4 == 2:
            cl.states["mem_free_mb"] = 1.0
        if seed % 4 == 3:
            cl.requests["slo_tbt_ms"] = 1e-3
        seen |= set(oracle.dispatch(cl.lat, cl.pow, cl.models, cl.states, cl.requests)["f_req"].tolist())
    assert seen == {1, 2, 3, -1}


def _toy(K, F=3, S=4, B=2, M=2):
    """Hand-filled LUT: every entry set explicitly by the test; model 0 is the request's model and is
    resident nowhere (all pairs cold, load_ms = 0), model 1 is the tenant of every GPU."""
    lat = np.ones((M, 2, F, S, B), dtype=f32); pw = np.ones_like(lat)
    models = np.zeros(M, dtype=synth.MODEL_INFO_DT); models["kv_mb_per_token"] = 1.0
    st = np.zeros(K, dtype=synth.GPU_STATE_DT)
    st["t"]["model"] = -1
    rq = np.zeros(1, dtype=synth.REQUEST_DT)
    rq["model"] = 0; rq["L"] = 1; rq["o_pred"] = 0; rq["slo_ttft_ms"] = 200.0; rq["slo_tbt_ms"] = 1e9
    return lat, pw, models, st, rq


def test_fig6_phase1_and_phase2():
    """Fig. 6: only GPUs whose estimated timestamp is below the SLO target of
    200 are feasible; among them the one with the lower energy (30 J) is selected.  Eq. 2 by hand:
    E^k = Power(f_k) x Latency(f_k, S_k, ...) read at each GPU's own frequency and free share."""
    lat, pw, models, st, rq = _toy(K=3)
    # GPU k: frequency index k, 2 share units taken -> SM_free = 2 -> sigma = 1
    for k, (t_avail, l, p) in enumerate([(100.0, 50.0, 900.0), (120.0, 60.0, 500.0), (150.0, 60.0, 100.0)]):
        _gpu(st, k, 1, 2, k, t_avail, 1e6)
        lat[0, 0, k, 1, 0] = l; pw[0, 0, k, 1, 0] = p      # batch bucket min(L,B)-1 = 0, rounds = 1
    o = oracle.dispatch(lat, pw, models, st, rq)[0]
    # timestamps 150, 180, 210: GPU 2 misses the SLO although it would be the cheapest (6 J)
    # energies: GPU 0 = 50 ms * 900 W = 45,000 mJ; GPU 1 = 60 ms * 500 W = 30,000 mJ  -> GPU 1
    assert (o["gpu"], o["sigma"], o["phi"], o["f_req"]) == (1, 1, 1, 1)
    assert o["energy_mj"] == f32(30000.0) and o["ttft_ms"] == f32(180.0)
    st["t_avail_ms"][2] = 139.0                             # now 199 < 200: the 6 J GPU wins
    o = oracle.dispatch(lat, pw, models, st, rq)[0]
    assert (o["gpu"], o["energy_mj"]) == (2, f32(6000.0))


def test_two_percent_band_tie_breaker():
    """within 2 % -> most free memory, then largest SM_free."""
    lat, pw, models, st, rq = _toy(K=3, F=1)
    for k, (l, smu, mem) in enumerate([(100.0, 2, 1000.0), (101.5, 2, 5000.0), (103.0, 2, 9000.0)]):
        _gpu(st, k, 1, smu, 0, 0.0, mem)
    lat[0, 0, 0, 1, 0] = 100.0
    o = oracle.dispatch(lat, pw, models, st, rq)[0]
    assert o["gpu"] == 2                                     # equal energies: the most free memory
    # separate the energies through the free share (sigma = SM_free - 1 indexes the LUT)
    lat2 = lat.copy()
    st2 = st.copy()
    _gpu(st2, 0, 1, 1, 0, 0.0, 1000.0)                       # SM_free 3 -> sigma 2
    _gpu(st2, 1, 1, 2, 0, 0.0, 5000.0)                       # SM_free 2 -> sigma 1
    _gpu(st2, 2, 1, 3, 0, 0.0, 9000.0)                       # SM_free 1 -> sigma 0
    lat2[0, 0, 0, 2, 0] = 100.0; lat2[0, 0, 0, 1, 0] = 101.5; lat2[0, 0, 0, 0, 0] = 103.0
    o = oracle.dispatch(lat2, pw, models, st2, rq)[0]
    assert o["gpu"] == 1 and o["energy_mj"] == f32(101.5)    # 101.5 <= 102: more free memory beats lower E
    lat2[0, 0, 0, 0, 0] = 101.9                              # GPU 2 enters the band with the most memory
    assert oracle.dispatch(lat2, pw, models, st2, rq)[0]["gpu"] == 2
    st2["mem_free_mb"] = 4000.0                              # equal memory: largest SM_free (GPU 0)
    assert oracle.dispatch(lat2, pw, models, st2, rq)[0]["gpu"] == 0


def test_phase3_fmax_retry_in_tavail_order_then_scale_out():
    """PAPER.md lines 231-233."""
    lat, pw, models, st, rq = _toy(K=3, F=3)
    for k, t_avail in enumerate([90.0, 50.0, 70.0]):
        _gpu(st, k, 1, 2, 0, t_avail, 1e6)                   # all at the lowest frequency
    lat[0, 0, 0, 1, 0] = 500.0                               # too slow at F_curr everywhere
    lat[0, 0, 2, 1, 0] = 120.0                               # at F_max: 210, 170, 190 -> GPUs 1 and 2 feasible
    pw[0, 0, 2, 1, 0] = 7.0
    o = oracle.dispatch(lat, pw, models, st, rq)[0]
    assert (o["gpu"], o["phi"], o["f_req"]) == (1, 2, 2)     # earliest T_avail among the feasible
    assert o["energy_mj"] == f32(840.0) and o["ttft_ms"] == f32(170.0)
    lat[0, 0, 2, 1, 0] = 160.0                               # nobody makes it: scale out
    lat[0, 0, :, 3, 0] = [400.0, 150.0, 100.0]               # fresh GPU, all 4 units (sigma 3), wait = load = 0
    pw[0, 0, :, 3, 0] = [1.0, 2.0, 5.0]                      # energies 400 (infeasible), 300, 500
    o = oracle.dispatch(lat, pw, models, st, rq)[0]
    assert (o["gpu"], o["sigma"], o["phi"], o["f_req"]) == (-1, 3, 1, 3) and o["energy_mj"] == f32(300.0)
    rq["slo_ttft_ms"] = 50.0
    o = oracle.dispatch(lat, pw, models, st, rq)[0]
    assert (o["gpu"], o["phi"], o["f_req"]) == (-1, -1, -1) and np.isinf(o["energy_mj"])
