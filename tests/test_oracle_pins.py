"""Pins of the CPU oracle against things other than itself (-m "not gpu").

Each test cites the passage (P:NNN = line of PAPER.md) or the mathematical fact it pins.
"""
from __future__ import annotations

import numpy as np
import pytest

import oracle
from paper_2606_30391_b200 import synth
import fs_brute as brute
from fs_util import (cluster_from, mk_models, mk_requests, mk_state, mk_states, tie_heavy)

f32 = np.float32
INF = np.float32(np.inf)


def _place(cl, nthreads=1):
    return oracle.place_batch(cl.lat, cl.pow, cl.models, cl.states, cl.requests, nthreads)


def _consol(cl):
    P = cl.params
    return oracle.consolidate(cl.lat, cl.pow, cl.models, cl.states, P.p_idle_w, P.horizon_ms,
                              P.mem_cap_mb, P.delta_pct)


# ---------------------------------------------------------------------------------------------
# slot rule: Energy = Power x Time (Eq. 1), deadline at a frequency
def test_slot_rule_by_hand():
    lat = np.zeros((1, 2, 1, 1, 4), dtype=np.float32)
    pw = np.zeros_like(lat)
    lat[0, 0, 0, 0, 3] = 12.5
    pw[0, 0, 0, 0, 3] = 200.0
    lat[0, 1, 0, 0, 1] = 30.0
    pw[0, 1, 0, 0, 1] = 150.0
    # prefill: 10 tokens in batches of 4 -> 3 rounds x 12.5 ms = 37.5 ms; 37.5 ms x 200 W = 7500 mJ
    ok, t, e = oracle.slot(lat, pw, 0, 0, 0, 0, 3, 10, 100.0, 137.5)
    assert ok and t == f32(37.5) and e == f32(7500.0)      # 100 + 37.5 <= 137.5 holds with equality
    ok, _, _ = oracle.slot(lat, pw, 0, 0, 0, 0, 3, 10, 100.0, 137.49)
    assert not ok
    # decode: 7 tokens in batches of 2 -> 4 rounds x 30 ms = 120 ms, 18000 mJ; deadline on ONE step
    ok, t, e = oracle.slot(lat, pw, 0, 1, 0, 0, 1, 7, 1e6, 30.0)
    assert ok and t == f32(120.0) and e == f32(18000.0)     # wait is ignored for TBT
    ok, _, _ = oracle.slot(lat, pw, 0, 1, 0, 0, 1, 7, 0.0, 29.9)
    assert not ok
    # empty queue costs nothing and is always feasible
    assert oracle.slot(lat, pw, 0, 0, 0, 0, 3, 0, 1e9, 0.0) == (True, f32(0), f32(0))


# ---------------------------------------------------------------------------------------------
# Eq. 2-3 and the Fig. 6 narrative: three GPUs, deadline 200; the GPU
# whose estimated completion exceeds 200 is dropped; of the two feasible ones the 30 J GPU wins.
def test_place_eq2_eq3_fig6_toy():
    M, F, S, B = 1, 1, 4, 1
    lat = np.zeros((M, 2, F, S, B), dtype=np.float32)
    pw = np.full_like(lat, 100.0)                     # 100 W everywhere
    lat[0, 0, 0, :, 0] = [60.0, 45.0, 30.0, 20.0]     # prefill ms per token at share 1/4..4/4
    lat[0, 1, 0, :, 0] = 1.0                          # decode unused (o_pred = 0)
    ten = dict(model=0, q=(0, 0))                     # co-resident with empty queues: A = Ecur = 0
    states = mk_states([
        mk_state(t_avail=0.0, tenants=[dict(ten, sigma=0)]),     # sm_free 3: grants 600/450/300 ms
        mk_state(t_avail=20.0, tenants=[dict(ten, sigma=1)]),    # sm_free 2: grants 600/450 ms
        mk_state(t_avail=150.0, tenants=[dict(ten, sigma=0)]),   # sm_free 3, but late
    ])
    # L = 10 tokens at batch bucket min(L,B)-1 = 0 -> 10 rounds; E = Power x Latency (Eq. 2):
    # 600 ms -> 60 J, 450 ms -> 45 J, 300 ms -> 30 J.
    reqs = mk_requests([dict(model=0, L=10, o_pred=0, ttft=500.0)])
    cl = cluster_from(lat, pw, mk_models(1), states, reqs)
    # deadline 500: GPU0 {45 J, 30 J}, GPU1 {20+450: 45 J}, GPU2 {150+300: 30 J}.  Eq. 3 picks
    # 30 J; the exact tie GPU0/GPU2 goes to the lowest flat index.
    out = _place(cl)[0]
    assert (out["gpu"], out["sigma"], out["phi"]) == (0, 2, 0)
    assert out["energy_mj"] == f32(30000.0) and out["ttft_ms"] == f32(300.0)
    assert out["flat"] == (0 * S + 2) * F + 0
    # deadline 400: Phase 1 drops GPU1 (470) and GPU2 (450); GPU0's 300 ms grant remains
    cl.requests["slo_ttft_ms"] = 400.0
    out = _place(cl)[0]
    assert (out["gpu"], out["sigma"], out["energy_mj"]) == (0, 2, f32(30000.0))
    # deadline 200: the candidate set is empty -> scale-out cue
    cl.requests["slo_ttft_ms"] = 200.0
    out = _place(cl)[0]
    assert out["gpu"] == -1 and out["phi"] == -1 and np.isinf(out["energy_mj"])
    # "the 30 J GPU wins": GPU0 has 1 free unit (60 J), GPU1 2 (45 J), GPU2 3 (30 J)
    cl.states[0]["t"][0]["sigma"] = 2
    cl.states[2]["t_avail_ms"] = 10.0
    cl.requests["slo_ttft_ms"] = 1000.0
    out = _place(cl)[0]
    assert (out["gpu"], out["sigma"], out["energy_mj"]) == (2, 2, f32(30000.0))
    assert out["ttft_ms"] == f32(310.0)
    cl.requests["slo_ttft_ms"] = 310.0                # equality still meets the deadline
    assert _place(cl)[0]["gpu"] == 2
    cl.requests["slo_ttft_ms"] = 309.9                # 10+300 > 309.9, 20+450, 600: nothing fits
    assert _place(cl)[0]["gpu"] == -1
    cl.requests["slo_ttft_ms"] = 470.0                # GPU1's 45 J grant fits exactly; GPU2 30 J wins
    assert _place(cl)[0]["gpu"] == 2
    cl.states[2]["mem_free_mb"] = 0.0                 # memory must fit
    cl.models["kv_mb_per_token"] = 1.0
    out = _place(cl)[0]
    assert (out["gpu"], out["sigma"], out["energy_mj"]) == (1, 1, f32(45000.0))


def test_place_energy_is_power_times_latency_when_coresidents_idle():
    """Eq. 2 special case: with idle co-residents dE is exactly the request's own
    Power x Latency summed over its two phases, and the answer is the table argmin (np.argmin)."""
    cl = synth.make_custom(seed=11, K=1, M=2, F=8, S=8, B=8, R=16, lo=1, hi=1)
    cl.states["t"]["q"][...] = 0
    cl.states["t"]["sigma"][...] = 0
    cl.states["t_avail_ms"] = 0
    cl.states["mem_free_mb"] = 1e9
    cl.models["load_ms"] = 0
    cl.requests["slo_ttft_ms"] = np.inf
    cl.requests["slo_tbt_ms"] = np.inf
    out = _place(cl)
    smf = cl.S - 1
    for r, rq in enumerate(cl.requests):
        m, L = int(rq["model"]), int(rq["L"])
        O = (21 * int(rq["o_pred"]) + 19) // 20
        b0 = min(L, cl.B) - 1
        r0 = -(-L // (b0 + 1))
        # planes [F][S] -> energy grid in fp32, vectorised (library ops, not the oracle's loops)
        e0 = (f32(r0) * cl.lat[m, 0, :, :, b0]) * cl.pow[m, 0, :, :, b0]
        e1 = (f32(O) * cl.lat[m, 1, :, :, 0]) * cl.pow[m, 1, :, :, 0]
        grid = (e0 + e1).T[:smf]                       # [sigma][phi], the flat order of one GPU
        idx = int(np.argmin(grid))                     # first minimum = lowest flat index
        assert out[r]["flat"] == idx and out[r]["energy_mj"] == grid.flat[idx]
        assert out[r]["f_req"] == 0                    # every frequency feasible (invariant v)


# ---------------------------------------------------------------------------------------------
# brute force on tiny clusters (independent numpy evaluator, all candidates enumerated)
def _check_place_against_brute(cl):
    out = _place(cl)
    n_feasible = 0
    for r in range(cl.R):
        b = brute.place_best(cl, r)
        o = out[r]
        if b is None:
            assert o["gpu"] == -1 and o["phi"] == -1 and o["sigma"] == -1 and np.isinf(o["energy_mj"])
            continue
        n_feasible += 1
        dE, flat, k, sg, phi, br1, ttft, tbt = b
        assert (o["gpu"], o["sigma"], o["phi"], o["beta"], o["flat"]) == (k, sg, phi, br1, flat), r
        assert o["energy_mj"] == f32(dE) and o["ttft_ms"] == ttft and o["tbt_ms"] == tbt
        # f_req: lowest feasible phi at the chosen (gpu, sigma)
        cands = brute.place_candidates(cl, r)
        assert o["f_req"] == min(c[4] for c in cands if c[2] == k and c[3] == sg)
    return n_feasible


@pytest.mark.parametrize("seed", range(24))
def test_place_bruteforce_tiny(seed):
    cl = synth.make_custom(seed=100 + seed, K=4, M=3, F=4, S=4, B=4, R=8, lo=1, hi=4)
    if seed % 3 == 1:      # stress the deadlines
        cl.requests["slo_ttft_ms"] *= 0.25
        cl.states["t"]["slo_ms"][...] *= 0.5
    if seed % 3 == 2:      # exact ties everywhere
        tie_heavy(cl, seed)
        cl.models["load_ms"] = 1.0
    _check_place_against_brute(cl)


def test_place_bruteforce_some_feasible_and_some_not():
    tot = feas = 0
    for seed in range(6):
        cl = synth.make_custom(seed=300 + seed, K=3, M=2, F=4, S=4, B=4, R=8, lo=1, hi=2)
        feas += _check_place_against_brute(cl)
        tot += cl.R
    assert 0 < feas < tot or feas == tot   # the pin must exercise real decisions
    assert feas > tot // 4


def test_place_tiny_config_sample_bruteforce():
    """BASELINE.json configs[0] (8 GPUs, 3 models, F=16, S=8, B=16): a sample of its requests."""
    cl = synth.make_cluster("tiny")
    full = _place(cl)
    sub = synth.make_cluster("tiny")
    sub.requests = cl.requests[:24].copy()
    out = _place(sub)
    assert np.array_equal(out, full[:24])
    for r in range(sub.R):
        b = brute.place_best(sub, r)
        if b is None:
            assert out[r]["gpu"] == -1
        else:
            assert (out[r]["flat"], out[r]["energy_mj"]) == (b[1], f32(b[0]))


def test_place_threads_do_not_change_results():
    cl = synth.make_cluster("tiny")
    assert np.array_equal(_place(cl, 1), _place(cl, 4))


# ---------------------------------------------------------------------------------------------
# tie rule (R:s6): exact ties go to the lowest flat index
def test_place_duplicate_gpu_and_duplicate_frequency():
    cl = synth.make_custom(seed=7, K=2, M=2, F=4, S=4, B=4, R=12, lo=1, hi=2)
    cl.states[1] = cl.states[0]                      # two identical GPUs -> GPU 0 wins
    out = _place(cl)
    assert np.all(out["gpu"] <= 0)
    assert np.any(out["gpu"] == 0)
    # duplicate frequency rows: phi=1 is a copy of phi=0, phi=3 a copy of phi=2 -> even phi only
    cl.lat[:, :, 1] = cl.lat[:, :, 0]
    cl.pow[:, :, 1] = cl.pow[:, :, 0]
    cl.lat[:, :, 3] = cl.lat[:, :, 2]
    cl.pow[:, :, 3] = cl.pow[:, :, 2]
    cl.states["f_cur"] = 0
    out = _place(cl)
    placed = out[out["gpu"] >= 0]
    assert len(placed) and np.all(placed["phi"] % 2 == 0) and np.all(placed["f_req"] % 2 == 0)


# ---------------------------------------------------------------------------------------------
# invariants (north star): frequency floor monotone in load; relaxing SLOs -> f_req == 0
def test_place_freq_floor_monotone_in_prompt_length():
    cl = synth.make_custom(seed=5, K=3, M=2, F=16, S=8, B=8, R=1, lo=1, hi=2)
    cl.states["mem_free_mb"] = 1e9
    cl.requests["slo_ttft_ms"] = 900.0
    base = cl.requests[0].copy()
    lens = [8, 16, 64, 256, 1024, 4096]
    for k in range(cl.K):                             # per GPU, per grant: f_req(L) non-decreasing
        one = synth.make_custom(seed=5, K=3, M=2, F=16, S=8, B=8, R=1, lo=1, hi=2)
        one.states = cl.states[k:k + 1].copy()
        one.K = 1
        prev = -1
        for L in lens:
            one.requests = np.array([base])
            one.requests["L"] = L
            one.requests["slo_ttft_ms"] = 900.0
            # candidates of every sigma via brute force; floor = min feasible phi over the grid
            c = brute.place_candidates(one, 0)
            if not c:
                prev = 10 ** 9                         # once infeasible, longer prompts stay so
                continue
            floor = min(x[4] for x in c)
            assert floor >= prev or prev == 10 ** 9
            assert prev != 10 ** 9
            prev = floor


def test_segmented_max_over_coresidents():
    """Device-wide operating point: the GPU's lowest feasible frequency is the max over
    co-residents of each one's lowest feasible frequency."""
    cl = synth.make_cluster("rack")
    seen = 0
    for k in range(cl.K):
        g = cl.states[k]
        fm = [oracle.tenant_fmin(cl.lat, cl.pow, g, i) for i in range(int(g["n_res"]))]
        floor = oracle.gpu_freq_floor(cl.lat, cl.pow, g)
        if min(fm) < 0:
            assert floor == -1
        else:
            assert floor == max(fm)          # tables are monotone in frequency
            seen += 1
        if g["n_res"] >= 2 and floor >= 0:   # removing a tenant never raises the floor
            h = g.copy()
            h["n_res"] -= 1
            assert 0 <= oracle.gpu_freq_floor(cl.lat, cl.pow, h) <= floor
    assert seen >= cl.K // 4


def test_place_continuous_optimum_of_generator():
    """Closed form: E(f) = rounds*tau*n^g*(a'/f + b)*(P_s + D f^3) is unimodal with optimum at
    2 D a' f^3 + 3 D b f^4 = P_s a'  (a' = a/s, D = 600 c s (0.3+0.7 n/B)); the discrete argmin
    must be a grid neighbour of it."""
    seed, M, F, S, B = 21, 4, 64, 8, 16
    cl = synth.make_custom(seed=seed, K=1, M=M, F=F, S=S, B=B, R=M, lo=1, hi=1)
    a, b, c, p_s = synth.table_coeffs(seed, M)
    cl.states["t"]["q"][...] = 0
    cl.states["t"]["sigma"][...] = S - 2              # sm_free = 1 -> grant sigma = 0 only
    cl.states["mem_free_mb"] = 1e9
    cl.requests["model"] = np.arange(M)
    cl.requests["L"] = 4 * B                          # bucket B-1, 4 rounds
    cl.requests["o_pred"] = 0                         # prefill only
    cl.requests["slo_ttft_ms"] = np.inf
    out = _place(cl)
    fh = cl.freq_mhz.astype(np.float64) / 1980.0
    for m in range(M):
        sh = 1.0 / S
        ap = a[m, 0] / sh
        D = 600.0 * c[m, 0] * sh * (0.3 + 0.7 * B / B)
        coeffs = [3 * D * b[m, 0], 2 * D * ap, 0, 0, -p_s[m] * ap]
        roots = [z.real for z in np.roots(coeffs) if abs(z.imag) < 1e-9 and z.real > 0]
        assert len(roots) == 1
        fstar = roots[0]
        phi = int(out[m]["phi"])
        lo = fh[max(phi - 1, 0)]
        hi = fh[min(phi + 1, F - 1)]
        assert lo <= fstar <= hi or (phi == F - 1 and fstar >= fh[-1]) or (phi == 0 and fstar <= fh[0])


# ---------------------------------------------------------------------------------------------
# local configuration: Fig. 8 step 3 worked table
def _fig8_cluster():
    # frequencies (900, 1100, 1300) MHz, S = 10 shares of 10 %, one batch level; four single-slot
    # tasks P1 (prefill), D1, D2, D3 (decode).  Minimum shares meeting the deadlines:
    #   900: (50,20,30,20) % = 120 %   1100: (40,20,20,20) % = 100 %   1300: (30,20,20,20) % = 90 %
    # and energies at those shares summing to 536 / 410 / 418 J.
    F, S = 3, 10
    lat = np.zeros((4, 2, F, S, 1), dtype=np.float32)
    pw = np.zeros_like(lat)
    min_units = {0: (5, 4, 3), 1: (2, 2, 2), 2: (3, 2, 2), 3: (2, 2, 2)}
    # P1: 10 prompt tokens, ms/token (100, 80, 50) at >= min share, W (230, 287.5, 458):
    #     230 J, 230 J, 229 J.  Below the minimum share it is 10x slower (misses TTFT 1500 ms).
    # Dx: 12 decode tokens, ms/step (50, 40, 35), W (170, 125, 150): 102 J, 60 J, 63 J.
    p_lat, p_pw = (100.0, 80.0, 50.0), (230.0, 287.5, 458.0)
    d_lat, d_pw = (50.0, 40.0, 35.0), (170.0, 125.0, 150.0)
    for m in range(4):
        ph = 0 if m == 0 else 1
        for phi in range(F):
            good_lat = p_lat[phi] if m == 0 else d_lat[phi]
            for sg in range(S):
                okk = sg + 1 >= min_units[m][phi]
                lat[m, ph, phi, sg, 0] = good_lat if okk else good_lat * 10.0
                pw[m, ph, phi, sg, 0] = p_pw[phi] if m == 0 else d_pw[phi]
        lat[m, 1 - ph] = 1.0
        pw[m, 1 - ph] = 1.0
    tenants = [dict(model=0, sigma=0, q=(10, 0), slo=(1500.0, 100.0))]
    tenants += [dict(model=m, sigma=0, q=(0, 12), slo=(1500.0, 100.0)) for m in (1, 2, 3)]
    states = mk_states([mk_state(tenants=tenants)])
    return cluster_from(lat, pw, mk_models(4), states, mk_requests([]))


def test_local_fig8_step3_worked_example():
    cl = _fig8_cluster()
    o = oracle.local_config(cl.lat, cl.pow, cl.states, oracle.OBJ_ENERGY | oracle.SPLIT_MINSM)[0]
    assert o["phi"] == 1                                        # 1100 MHz is chosen
    assert tuple(o["sigma"]) == (3, 1, 1, 1)                    # 40/20/20/20 % (index = units-1)
    assert o["cost"] == f32(410000.0) and o["energy_mj"] == f32(410000.0)   # 410 J
    assert o["f_req"] == 1                                      # 900 MHz needs 120 % -> infeasible
    # the 1300 MHz row: feasible with 90 % and 418 J; forbid 1100 MHz and it must be chosen
    cl.lat[:, :, 1] *= 100.0
    o = oracle.local_config(cl.lat, cl.pow, cl.states, oracle.OBJ_ENERGY | oracle.SPLIT_MINSM)[0]
    assert o["phi"] == 2 and tuple(o["sigma"]) == (2, 1, 1, 1) and o["cost"] == f32(418000.0)
    # the 900 MHz row's 536 J: allow 120 % by giving the GPU 12 share units
    cl2 = _fig8_cluster()
    lat12 = np.concatenate([cl2.lat, cl2.lat[:, :, :, -2:]], axis=3)
    pw12 = np.concatenate([cl2.pow, cl2.pow[:, :, :, -2:]], axis=3)
    o = oracle.local_config(np.ascontiguousarray(lat12[:, :, :1]), np.ascontiguousarray(pw12[:, :, :1]),
                            cl2.states, oracle.OBJ_ENERGY | oracle.SPLIT_MINSM)[0]
    assert o["phi"] == 0 and tuple(o["sigma"]) == (4, 1, 2, 1) and o["cost"] == f32(536000.0)


@pytest.mark.parametrize("seed", range(12))
@pytest.mark.parametrize("flags", [0, 1, 2, 3])
def test_local_bruteforce_tiny(seed, flags):
    cl = synth.make_custom(seed=400 + seed, K=3, M=4, F=4, S=5, B=6, R=0, lo=1, hi=4,
                           local_sweep=(seed % 2 == 0))
    if seed % 2 == 0:
        cl.states["t"]["q"][...] = np.minimum(cl.states["t"]["q"], 9)
    if seed % 3 == 2:
        tie_heavy(cl, seed)
    cl.states["t"]["slo_ms"][..., 0] *= 0.05 if seed % 2 else 1.0
    out = oracle.local_config(cl.lat, cl.pow, cl.states, flags)
    for k in range(cl.K):
        b = brute.local_best(cl, k, bool(flags & 1), bool(flags & 2))
        o = out[k]
        n = int(cl.states[k]["n_res"])
        if b is None:
            assert o["phi"] == -1 and np.isinf(o["cost"])
            continue
        (C, flat), phi, sp, betas = b
        assert (o["phi"], o["flat"]) == (phi, flat) and o["cost"] == f32(C)
        assert tuple(o["sigma"][:n]) == tuple(sp)
        assert [tuple(x) for x in o["beta"][:n]] == [tuple(x) for x in betas]


def test_local_freq_floor_same_in_both_split_modes():
    """Tables monotone in sigma => a frequency has a feasible split with sum == S iff the
    minimum shares fit (sum <= S): f_req agrees between EXHAUSTIVE and MINSM."""
    cl = synth.make_custom(seed=31, K=32, M=8, F=16, S=8, B=16, R=0, lo=2, hi=4, local_sweep=True)
    a = oracle.local_config(cl.lat, cl.pow, cl.states, oracle.SPLIT_EXHAUSTIVE)
    b = oracle.local_config(cl.lat, cl.pow, cl.states, oracle.SPLIT_MINSM)
    assert np.array_equal(a["f_req"], b["f_req"])
    assert np.any(a["f_req"] > 0) and np.any(a["phi"] >= 0)
    # EXHAUSTIVE searches a superset of sigma-tuples at sum == S ... its optimum is never worse
    ok = (a["phi"] >= 0) & (b["phi"] >= 0)
    full = np.array([sum(int(s) + 1 for s in o["sigma"][:int(n)]) == cl.S
                     for o, n in zip(b, cl.states["n_res"])])
    assert np.all(a["cost"][ok & full] <= b["cost"][ok & full])


def test_local_inactive_gpu():
    cl = _fig8_cluster()
    cl.states["n_res"] = 0
    o = oracle.local_config(cl.lat, cl.pow, cl.states, 0)[0]
    assert o["phi"] == -1 and o["cost"] == 0


# ---------------------------------------------------------------------------------------------
# consolidation
@pytest.mark.parametrize("seed", range(10))
def test_consolidate_bruteforce_tiny(seed):
    cl = synth.make_custom(seed=500 + seed, K=6, M=5, F=4, S=8, B=4, R=0, lo=1, hi=2,
                           profile="beta25")
    cl.states["t"]["mem_used_mb"][...] *= 0.5
    if seed % 3 == 2:
        tie_heavy(cl, seed)
    if seed == 4:
        cl.states[2]["n_res"] = 0
    out = _consol(cl)
    ref = brute.consolidate_all(cl)
    P = cl.params
    n_dst = 0
    for a in range(cl.K):
        dst, phi, score, cstar_a = ref[a]
        o = out[a]
        assert (o["dst"], o["phi"]) == (dst, phi)
        if dst < 0:
            assert np.isinf(o["score_mj"]) and o["saving_mj"] == -np.inf
            continue
        n_dst += 1
        assert o["score_mj"] == score
        na = int(cl.states[a]["n_res"])
        mig = f32(0)
        for i in range(na):
            v = cl.models["mig_mj"][int(cl.states[a]["t"][i]["model"])]
            mig = v if i == 0 else f32(mig + v)
        want = f32(f32(f32(f32(P.p_idle_w) * f32(P.horizon_ms)) + cstar_a) - f32(score + mig))
        assert o["saving_mj"] == want
    assert n_dst > 0 or seed in ()


def test_consolidate_pair_cost_is_symmetric_and_empty_destination():
    # two GPUs with one tenant each; C*_ab == C*_ba (fp32 addition commutes, constraints symmetric)
    cl = synth.make_custom(seed=611, K=2, M=4, F=8, S=8, B=4, R=0, lo=1, hi=1, profile="beta25")
    cl.states["t"]["mem_used_mb"][...] = 100.0
    out = _consol(cl)
    ref = brute.consolidate_all(cl)
    if out[0]["dst"] == 1 and out[1]["dst"] == 0:
        cab = f32(out[0]["score_mj"] + ref[1][3])
        cba = f32(out[1]["score_mj"] + ref[0][3])
        # score = C*_ab - C*_b, so C*_ab is recovered up to one rounding; compare the phi instead
        assert out[0]["phi"] == out[1]["phi"]
        assert abs(float(cab) - float(cba)) <= 4e-7 * abs(float(cab)) + 1e-3
    # destination with empty queues: E_b == 0, C*_b == 0  =>  score(a->b) == C*_a when the SM
    # cap does not bind
    cl.states[1]["t"]["q"][...] = 0
    out = _consol(cl)
    ref = brute.consolidate_all(cl)
    assert out[0]["dst"] == 1
    assert out[0]["score_mj"] == ref[0][3]            # == C*_a
    assert out[1]["score_mj"] == ref[0][3] - 0 or out[1]["dst"] == 0


def test_consolidate_appendix_g_arithmetic():
    """disabling one GPU for 5 min saves 29.6 kJ; migrating Llama2-13B costs 10.67 J
    (recovered after 108 ms), Qwen3-32B 40.76 J (413 ms)."""
    # idle power implied by the paper: 29.6 kJ / 300 s = 98.67 W; recovery times check
    assert round(10.67 / 98.67 * 1000) == 108 and round(40.76 / 98.67 * 1000) == 413
    lat = np.ones((2, 2, 2, 4, 2), dtype=np.float32)
    pw = np.ones_like(lat)
    models = mk_models(2)
    models["mig_mj"] = [10670.0, 40760.0]
    idle = dict(q=(0, 0), mem=10.0)
    states = mk_states([mk_state(tenants=[dict(idle, model=0)]), mk_state(tenants=[dict(idle, model=1)])])
    cl = cluster_from(lat, pw, models, states, mk_requests([]),
                      synth.Params(p_idle_w=98.67, horizon_ms=300000.0, mem_cap_mb=80000.0, delta_pct=5))
    out = _consol(cl)
    # idle term 98.67 W x 300,000 ms = 29,601,000 mJ (the paper's 29.6 kJ); zero dynamic terms
    assert out[0]["dst"] == 1 and out[0]["score_mj"] == 0
    assert out[0]["saving_mj"] == f32(29601000.0 - 10670.0)
    assert out[1]["saving_mj"] == f32(29601000.0 - 40760.0)
    # idle/migration ratios: the paper prints 2788x / 727x; 29,600/40.76 = 726.2, 29,600/10.67 = 2774
    assert abs(29600.0 / 40.76 - 727) < 1.0 and abs(29600.0 / 10.67 - 2774) < 1.0


def test_consolidate_margin_delta():
    """5 % safety margin on SMs and memory: S_eff = floor(0.95 S), M_eff = 0.95 cap."""
    lat = np.ones((2, 2, 1, 16, 1), dtype=np.float32)
    pw = np.ones_like(lat)
    # each tenant needs exactly 8 of 16 units at the only frequency: 8+8 = 16 > S_eff = 15
    lat[:, 1, 0, :7, 0] = 1000.0
    t = dict(q=(0, 5), slo=(1e9, 10.0), mem=100.0)
    states = mk_states([mk_state(tenants=[dict(t, model=0)]), mk_state(tenants=[dict(t, model=1)])])
    cl = cluster_from(lat, pw, mk_models(2), states, mk_requests([]))
    assert np.all(_consol(cl)["dst"] == -1)
    cl.params.delta_pct = 0                            # without the margin the pair fits
    assert np.all(_consol(cl)["dst"] >= 0)
    cl.params.delta_pct = 5
    lat[:, 1, 0, 6, 0] = 1.0                           # 7+7 = 14 <= 15 fits
    assert np.all(_consol(cl)["dst"] >= 0)
    cl.states["t"]["mem_used_mb"][...] = 38001.0       # 76,002 > 0.95 * 80,000 = 76,000
    assert np.all(_consol(cl)["dst"] == -1)
    cl.states["t"]["mem_used_mb"][...] = 38000.0
    assert np.all(_consol(cl)["dst"] >= 0)


# ---------------------------------------------------------------------------------------------
# Pair score with BUSY destinations, BY HAND (SURVEY 8(c) fs_consolidate steps 1-4; P:46, P:351, P:623;
# DESIGN s18 "score = extra energy the destination pays").  Six GPUs, F = 2, S = 16 (S_eff = 15), B = 2.
# Every tenant has an empty prefill queue and 4 decode tokens at bucket beta = 1: 2 rounds x LAT 2.0 = 4 ms,
# energy = 4 x POW.  A model's table makes it infeasible (LAT 1000 > TBT slack 10) below its minimum share and
# sets POW = E/4 there (E/8 at larger shares: the rule takes the LOWEST feasible share, not the cheapest).
#
#   GPU  tenants (model)   need[phi0, phi1]   E[phi0, phi1]     C*_g (own optimum)      sum of mig_mj
#   0    2 (0, 1)          4+4, 2+2 = 8, 4    100+50, 300+100   150  at phi 0           30+12 = 42
#   1    1 (2)             8, 3               1000, 1500        1000 at phi 0           5
#   2    1 (3)             8, 1               200, 800          200  at phi 0           7
#   3    1 (4)             8, 1               5000, 5100        5000 at phi 0           9
#   4    3 (5, 5, 5)       3, 3               3, 3              3    at phi 0 (tie)     6
#   5    1 (6)             8, 2               7000, 7100        7000 at phi 0           11
#
# Source 0 (2 tenants): GPU 4 is out (2 + 3 > 4 tenants) although it would score 153 - 3 = 150.  With every other
# destination phi 0 needs 8 + 8 = 16 > 15 units, so the merged GPU runs at phi 1 although BOTH run at phi 0 alone:
#   b=1: 1500+400 = 1900 - 1000 = 900     b=2: 800+400 = 1200 - 200 = 1000    (lowest C*_ab, not the lowest score)
#   b=3: 5100+400 = 5500 - 5000 = 500     b=5: 7100+400 = 7500 - 7000 = 500   (exact tie: lower index wins)
#   => dst 3, phi 1, score 500, saving = (100 W x 1000 ms + 150) - (500 + 42) = 99608.
# Source 1: b=0: 400+1500 - 150 = 1750; b=2: 2300 - 200 = 2100; b=3: 6600 - 5000 = 1600; b=5: 8600 - 7000 = 1600;
#   b=4 (1 + 3 = 4 tenants: allowed): phi 0 needs 8 + 3 = 11: 3 + 1000 = 1003 - 3 = 1000 => dst 4, phi 0,
#   saving = 101000 - (1000 + 5) = 99995.
# Source 4 (3 tenants: only single-tenant destinations): every one of b = 1, 2, 3, 5 costs E_b[0] + 3 - C*_b = 3
#   => dst 1, phi 0, saving = 100003 - (3 + 6) = 99994.
# Sources 2, 3, 5 all go to GPU 4 at phi 0: scores 203-3 = 200, 5003-3 = 5000, 7003-3 = 7000;
#   savings 100200 - 207 = 99993, 105000 - 5009 = 99991, 107000 - 7011 = 99989.
CONSOL_BY_HAND = [  # (dst, phi, score_mj, saving_mj) per source
    (3, 1, 500.0, 99608.0), (4, 0, 1000.0, 99995.0), (4, 0, 200.0, 99993.0),
    (4, 0, 5000.0, 99991.0), (1, 0, 3.0, 99994.0), (4, 0, 7000.0, 99989.0)]


def _consol_busy_cluster():
    need = {0: (4, 2), 1: (4, 2), 2: (8, 3), 3: (8, 1), 4: (8, 1), 5: (1, 1), 6: (8, 2)}
    energy = {0: (100, 300), 1: (50, 100), 2: (1000, 1500), 3: (200, 800), 4: (5000, 5100), 5: (1, 1), 6: (7000, 7100)}
    M, F, S, B = 7, 2, 16, 2
    lat = np.full((M, 2, F, S, B), 3.0, dtype=np.float32)       # bucket 0 and the prefill phase: never read
    pw = np.full((M, 2, F, S, B), 7.0, dtype=np.float32)
    for m in range(M):
        for phi in range(F):
            lo = need[m][phi] - 1
            lat[m, 1, phi, :lo, 1] = 1000.0
            lat[m, 1, phi, lo:, 1] = 2.0
            pw[m, 1, phi, :, 1] = energy[m][phi] / 8.0
            pw[m, 1, phi, lo, 1] = energy[m][phi] / 4.0
    models = mk_models(M)
    models["mig_mj"] = [30.0, 12.0, 5.0, 7.0, 9.0, 2.0, 11.0]
    t = lambda m, sg: dict(model=m, sigma=sg, beta=(0, 1), q=(0, 4), slo=(1e9, 10.0), mem=100.0)
    states = mk_states([mk_state(tenants=[t(0, 5), t(1, 5)]), mk_state(tenants=[t(2, 9)]), mk_state(tenants=[t(3, 9)]),
                        mk_state(tenants=[t(4, 9)]), mk_state(tenants=[t(5, 1), t(5, 1), t(5, 1)]), mk_state(tenants=[t(6, 9)])])
    return cluster_from(lat, pw, models, states, mk_requests([]),
                        synth.Params(p_idle_w=100.0, horizon_ms=1000.0, mem_cap_mb=80000.0, delta_pct=5))


def test_consolidate_busy_destinations_by_hand():
    out = _consol(_consol_busy_cluster())
    for a, (dst, phi, score, saving) in enumerate(CONSOL_BY_HAND):
        assert (int(out[a]["dst"]), int(out[a]["phi"])) == (dst, phi), a
        assert out[a]["score_mj"] == f32(score) and out[a]["saving_mj"] == f32(saving), a


# ---------------------------------------------------------------------------------------------
# Co-resident coupling BY HAND (P:44, P:127, P:265 shared operating point; DESIGN s4): a busy tenant of the
# request's model (bump: its decode batch grows by the new sequence) and a busy tenant of another model.
# Every number below is written out; none comes from fs_brute or from the oracle.
def _coupled_cluster(beta1=0, q1=4, tenant0_tbt=1e9):
    M, F, S, B = 2, 2, 4, 3
    lat = np.full((M, 2, F, S, B), 1000.0, dtype=np.float32)
    pw = np.full((M, 2, F, S, B), 1000.0, dtype=np.float32)
    # model 0, decode, share sigma=0 (tenant 0's share; also the request's grant sigma=0)
    lat[0, 1, 0, 0, 0], pw[0, 1, 0, 0, 0] = 10.0, 100.0     # phi 0, batch 1
    lat[0, 1, 1, 0, 0], pw[0, 1, 1, 0, 0] = 5.0, 300.0      # phi 1, batch 1
    lat[0, 1, 0, 0, 1], pw[0, 1, 0, 0, 1] = 12.0, 110.0     # phi 0, batch 2 (after the bump)
    lat[0, 1, 1, 0, 1], pw[0, 1, 1, 0, 1] = 6.0, 320.0      # phi 1, batch 2
    # model 0, decode, grant sigma=1
    lat[0, 1, 0, 1, 1], pw[0, 1, 0, 1, 1] = 8.0, 120.0
    lat[0, 1, 1, 1, 1], pw[0, 1, 1, 1, 1] = 4.0, 330.0
    lat[0, 1, 0, 1, 0], pw[0, 1, 0, 1, 0] = 7.0, 105.0      # batch 1 at sigma=1 (the no-bump twin)
    lat[0, 1, 1, 1, 0], pw[0, 1, 1, 1, 0] = 3.5, 310.0
    # model 0, prefill at batch bucket min(L,B)-1 = 1
    lat[0, 0, 0, 0, 1], pw[0, 0, 0, 0, 1] = 30.0, 100.0
    lat[0, 0, 1, 0, 1], pw[0, 0, 1, 0, 1] = 15.0, 250.0
    lat[0, 0, 0, 1, 1], pw[0, 0, 0, 1, 1] = 18.0, 120.0
    lat[0, 0, 1, 1, 1], pw[0, 0, 1, 1, 1] = 9.0, 260.0
    # model 1 (the other tenant), prefill, its share sigma=0, batch bucket 1
    lat[1, 0, 0, 0, 1], pw[1, 0, 0, 0, 1] = 20.0, 50.0
    lat[1, 0, 1, 0, 1], pw[1, 0, 1, 0, 1] = 10.0, 200.0
    tenants = [dict(model=0, sigma=0, beta=(0, beta1), q=(0, q1), slo=(1e9, tenant0_tbt)),
               dict(model=1, sigma=0, beta=(1, 0), q=(6, 0), slo=(1e9, 1e9))]
    states = mk_states([mk_state(f_cur=1, t_avail=7.0, tenants=tenants)])
    reqs = mk_requests([dict(model=0, L=2, o_pred=3)])       # O = ceil(1.05*3) = 4
    return cluster_from(lat, pw, mk_models(M), states, reqs)


def test_place_busy_coresidents_bump_and_negative_marginal_energy_by_hand():
    """GPU now (F_curr = phi 1, nobody bumped): tenant 0 decodes 4 tokens one by one, 4 x 5 ms x 300 W = 6000 mJ;
    tenant 1 prefills 6 tokens in batches of 2, 3 x 10 ms x 200 W = 6000 mJ: Ecur = 12000 mJ.
    After the request joins tenant 0's decode batch (batch 2: 2 rounds) the co-residents cost
      phi 0: 2 x 12 x 110 + 3 x 20 x 50 = 2640 + 3000 = 5640      phi 1: 2 x 6 x 320 + 3 x 10 x 200 = 9840
    and the request itself (prefill 1 round of 2 tokens; decode O = 4 in its tenant's batch 2: 2 rounds)
      (sigma 0, phi 0): 30 x 100 + 2 x 12 x 110 = 5640            (sigma 0, phi 1): 15 x 250 + 2 x 6 x 320 = 7590
      (sigma 1, phi 0): 18 x 120 + 2 x 8 x 120 = 4080             (sigma 1, phi 1): 9 x 260 + 2 x 4 x 330 = 4980
    dE = (A + e_r) - Ecur:  -720, 5430, -2280, 2820  ->  (sigma 1, phi 0) with a NEGATIVE marginal energy."""
    cl = _coupled_cluster()
    o = _place(cl)[0]
    assert (o["gpu"], o["sigma"], o["phi"], o["beta"], o["f_req"]) == (0, 1, 0, 1, 0)
    assert o["energy_mj"] == f32(-2280.0) and o["flat"] == (0 * 4 + 1) * 2 + 0
    assert o["ttft_ms"] == f32(25.0) and o["tbt_ms"] == f32(8.0)        # 7 + 18; LAT1 at the chosen point
    # request TBT SLO 7 ms: LAT1 = 12 / 8 at phi 0 miss it, 6 / 4 at phi 1 meet it -> (sigma 1, phi 1), 2820
    cl.requests["slo_tbt_ms"] = 7.0
    o = _place(cl)[0]
    assert (o["sigma"], o["phi"], o["f_req"]) == (1, 1, 1) and o["energy_mj"] == f32(2820.0)
    # request TTFT SLO 24 ms: 7+30, 7+18 miss, 7+15, 7+9 meet -> phi 1 again, (sigma 1) 2820
    cl.requests["slo_tbt_ms"] = 1e9
    cl.requests["slo_ttft_ms"] = 24.0
    o = _place(cl)[0]
    assert (o["sigma"], o["phi"]) == (1, 1) and o["ttft_ms"] == f32(16.0)
    # the bump also decides the co-resident's own deadline: tenant 0 must keep TBT <= 11 ms; alone it runs at
    # 10 ms (phi 0) but in batch 2 at 12 ms -> phi 0 is out for everyone (shared operating point)
    cl = _coupled_cluster(tenant0_tbt=11.0)
    o = _place(cl)[0]
    assert (o["sigma"], o["phi"], o["f_req"]) == (1, 1, 1) and o["energy_mj"] == f32(2820.0)


def test_place_bump_past_the_last_batch_level_drops_the_gpu():
    """beta_1 = B-1: one more sequence does not fit the profiled batch range -> not a candidate (DESIGN s4)."""
    cl = _coupled_cluster(beta1=2)
    o = _place(cl)[0]
    assert o["gpu"] == -1 and np.isinf(o["energy_mj"])


def test_place_idle_decode_queue_means_no_bump():
    """q_1 = 0: tenant 0 costs nothing now or later, the request opens batch 1 (bucket 0, 4 rounds):
      Ecur = 0 + 6000;  A = (0 + 3000, 0 + 6000)
      (0,0): 3000 + 4x10x100 = 7000 -> +3000 - 6000 = 4000      (0,1): 3750 + 4x5x300 = 9750 -> 9750
      (1,0): 2160 + 4x7x105 = 5100 -> 2100                      (1,1): 2340 + 4x3.5x310 = 6680 -> 6680"""
    cl = _coupled_cluster(q1=0)
    o = _place(cl)[0]
    assert (o["sigma"], o["phi"], o["beta"]) == (1, 0, 0)
    assert o["energy_mj"] == f32(2100.0) and o["tbt_ms"] == f32(7.0)


def test_place_cold_start_pays_the_weight_load():
    """A GPU that does not host the model adds load_ms to the request's wait: 10 + 100 + 50 = 160 ms."""
    M, F, S, B = 2, 1, 2, 1
    lat = np.ones((M, 2, F, S, B), dtype=np.float32)
    pw = np.ones_like(lat)
    lat[1, 0, 0, 0, 0], pw[1, 0, 0, 0, 0] = 50.0, 10.0       # request's prefill on one share unit: 50 ms, 500 mJ
    idle = dict(sigma=0, q=(0, 0))
    states = mk_states([mk_state(t_avail=10.0, tenants=[dict(idle, model=0)]),    # cold for model 1
                        mk_state(t_avail=130.0, tenants=[dict(idle, model=1)])])  # warm, but late: 130 + 50
    reqs = mk_requests([dict(model=1, L=1, o_pred=0, ttft=160.0)])
    cl = cluster_from(lat, pw, mk_models(M, load_ms=100.0), states, reqs)
    o = _place(cl)[0]
    assert o["gpu"] == 0 and o["ttft_ms"] == f32(160.0) and o["energy_mj"] == f32(500.0)
    cl.requests["slo_ttft_ms"] = 159.0                        # would pass without the load (60 ms): it must not
    assert _place(cl)[0]["gpu"] == -1
    cl.requests["slo_ttft_ms"] = 180.0                        # both feasible, equal energy: lowest flat index
    assert _place(cl)[0]["gpu"] == 0
    cl.states[0]["mem_free_mb"] = -1.0
    o = _place(cl)[0]
    assert o["gpu"] == 1 and o["ttft_ms"] == f32(180.0)       # warm: no load added


# ---------------------------------------------------------------------------------------------
# FS_OBJ_POWER by hand on a 2 x 2 x 3 table (F, S, B) ("minimum-power feasible config", configs[3])
def _power_cluster():
    F, S, B = 2, 2, 3
    lat = np.zeros((1, 2, F, S, B), dtype=np.float32)
    pw = np.zeros_like(lat)
    # prefill queue of 3 tokens (rounds 3, 2, 1 at batch 1, 2, 3), TTFT slack 100 ms
    lat[0, 0, 0, 0], pw[0, 0, 0, 0] = (40, 60, 120), (50, 45, 40)      # 120 ms at every batch: misses
    lat[0, 0, 0, 1], pw[0, 0, 0, 1] = (30, 45, 98), (70, 66, 62)       # 90 / 90 / 98 ms
    lat[0, 0, 1, 0], pw[0, 0, 1, 0] = (20, 30, 70), (120, 110, 130)    # 60 / 60 / 70 ms
    lat[0, 0, 1, 1], pw[0, 0, 1, 1] = (10, 15, 35), (200, 190, 210)
    # decode queue of 2 tokens (rounds 2, 1 at batch 1, 2; batch 3 > q is not a candidate), TBT slack 25 ms
    lat[0, 1, 0, 0], pw[0, 1, 0, 0] = (20, 24, 1), (30, 35, 1)
    lat[0, 1, 0, 1], pw[0, 1, 0, 1] = (15, 26, 1), (40, 20, 1)         # batch 2 is cheaper but misses 25 ms
    lat[0, 1, 1, 0], pw[0, 1, 1, 0] = (10, 12, 1), (90, 80, 1)
    lat[0, 1, 1, 1], pw[0, 1, 1, 1] = (5, 6, 1), (150, 140, 1)
    states = mk_states([mk_state(tenants=[dict(model=0, sigma=0, q=(3, 2), slo=(100.0, 25.0))])])
    return cluster_from(lat, pw, mk_models(1), states, mk_requests([]))


def test_local_power_objective_by_hand():
    cl = _power_cluster()
    # minimum-SM rule, POWER: phi 0 needs share 2/2 (share 1/2 misses TTFT): 62 W (batch 3) + 40 W (batch 1) = 102 W;
    # phi 1 runs on share 1/2: 110 W (batch 2) + 80 W (batch 2) = 190 W.  -> phi 0, 102 W, beta (2, 0);
    # energy there = 98 x 62 + 2 x 15 x 40 = 6076 + 1200 = 7276 mJ
    o = oracle.local_config(cl.lat, cl.pow, cl.states, oracle.OBJ_POWER | oracle.SPLIT_MINSM)[0]
    assert (o["phi"], o["f_req"], o["sigma"][0]) == (0, 0, 1) and tuple(o["beta"][0]) == (2, 0)
    assert o["cost"] == f32(102.0) and o["power_w"] == f32(102.0) and o["energy_mj"] == f32(7276.0)
    # ENERGY on the same input picks batch 2 for the prefill: 2 x 45 x 66 = 5940 (< 6300, 6076) + 1200 = 7140 mJ
    # against phi 1: min(7200, 6600, 9100) + min(1800, 960) = 7560 mJ; power there 66 + 40 = 106 W
    o = oracle.local_config(cl.lat, cl.pow, cl.states, oracle.OBJ_ENERGY | oracle.SPLIT_MINSM)[0]
    assert (o["phi"], o["sigma"][0]) == (0, 1) and tuple(o["beta"][0]) == (1, 0)
    assert o["cost"] == f32(7140.0) and o["energy_mj"] == f32(7140.0) and o["power_w"] == f32(106.0)
    # all splits summing to S: one tenant takes both units; phi 1 there costs 190 + 140 = 330 W -> phi 0 again
    o = oracle.local_config(cl.lat, cl.pow, cl.states, oracle.OBJ_POWER | oracle.SPLIT_EXHAUSTIVE)[0]
    assert (o["phi"], o["sigma"][0], o["flat"]) == (0, 1, 0) and o["cost"] == f32(102.0)
    # tighten the TTFT slack to 95 ms: batch 3 at phi 0 (98 ms) drops out -> 66 W (batch 2) + 40 W = 106 W
    cl.states[0]["t"][0]["slo_ms"][0] = 95.0
    o = oracle.local_config(cl.lat, cl.pow, cl.states, oracle.OBJ_POWER | oracle.SPLIT_MINSM)[0]
    assert o["cost"] == f32(106.0) and tuple(o["beta"][0]) == (1, 0)
    # 85 ms: phi 0 is infeasible at every share and batch -> phi 1 on share 1/2, 190 W; f_req = 1
    cl.states[0]["t"][0]["slo_ms"][0] = 85.0
    o = oracle.local_config(cl.lat, cl.pow, cl.states, oracle.OBJ_POWER | oracle.SPLIT_MINSM)[0]
    assert (o["phi"], o["f_req"], o["sigma"][0]) == (1, 1, 0) and o["cost"] == f32(190.0)
    assert tuple(o["beta"][0]) == (1, 1) and o["energy_mj"] == f32(2 * 30 * 110 + 12 * 80)
