"""Pins of the oracle's sequential commit pass between the requests of one batch (
DESIGN.md reading s34 of PAPER.md lines 214-218: a dispatched request starts at T_avail with all of
SM_free and holds it until it completes).  CPU only."""
from __future__ import annotations

import types

import numpy as np
import pytest

import oracle
from fs_brute import f32
from paper_2606_30391_b200 import synth
from test_oracle_dispatch import _gpu, _restate, _toy


def test_commit_by_hand():
    """Two GPUs, three identical requests.  GPU 0 is the cheaper one, so a snapshot dispatcher sends all
    three there; with the commit pass its T_avail moves to each request's completion time and the third
    request no longer meets the 200 ms target there."""
    lat, pw, models, st, rq = _toy(K=2, F=2)
    rq = np.repeat(rq, 4); rq["o_pred"] = 20                  # O = ceil(1.05 * 20) = 21 tokens, Req_mem = 22 MB
    for k, (t_avail, p) in enumerate([(10.0, 1.0), (0.0, 2.0)]):
        _gpu(st, k, 1, 2, 0, t_avail, 1000.0)                 # SM_free 2 -> sigma 1, F_curr = 0
    lat[0, 0, 0, 1, 0] = 50.0; lat[0, 1, 0, 1, 0] = 2.0       # prefill 50 ms, 21 decode rounds of 2 ms
    pw[0, :, 0, 1, 0] = 1.0
    lat[0, 0, 1, 1, 0] = 20.0; lat[0, 1, 1, 1, 0] = 1.0; pw[0, :, 1, 1, 0] = 9.0   # F_max: faster, dearer
    st["mem_free_mb"][1] = 500.0                              # GPU 0 has the most memory: it wins exact ties
    snap = oracle.dispatch(lat, pw, models, st, rq)
    assert snap["gpu"].tolist() == [0, 0, 0, 0]
    got, after = oracle.dispatch_commit(lat, pw, models, st, rq)
    # r0: GPU 0, ttft 10+50 = 60, done at 60+42 = 102.  r1: ttft 152, done 194.  r2: 194+50 > 200 on GPU 0 ->
    # GPU 1: ttft 50, done 92.  r3: GPU 0 still out, GPU 1: ttft 142, done 184.
    assert got["gpu"].tolist() == [0, 0, 1, 1] and got["f_req"].tolist() == [1, 1, 1, 1]
    assert got["ttft_ms"].tolist() == [60.0, 152.0, 50.0, 142.0]
    assert after["t_avail_ms"].tolist() == [194.0, 184.0]
    assert after["mem_free_mb"].tolist() == [1000.0 - 44.0, 500.0 - 44.0]
    assert after["f_cur"].tolist() == [0, 0]
    # a fifth request: nobody makes 200 ms at F_curr (244, 234); at F_max GPU 1 (earliest T_avail) does:
    # 184 + 20 = 204 > 200 no; GPU 0: 194 + 20 = 214 no -> scale-out, and no record changes
    got5, after5 = oracle.dispatch_commit(lat, pw, models, after, rq[:1])
    assert got5["gpu"][0] == -1 and got5["f_req"][0] == 3
    assert after5.tobytes() == after.tobytes()
    # with a 210 ms target the F_max retry takes GPU 1 (T_avail 184 < 194) and leaves it at F_max
    rq["slo_ttft_ms"] = 210.0
    got6, after6 = oracle.dispatch_commit(lat, pw, models, after, rq[:1])
    assert (got6["gpu"][0], got6["phi"][0], got6["f_req"][0], got6["ttft_ms"][0]) == (1, 1, 2, 204.0)
    assert after6["f_cur"].tolist() == [0, 1] and after6["t_avail_ms"].tolist() == [194.0, 204.0 + 21.0]
    assert after6["mem_free_mb"].tolist() == [956.0, 456.0 - 22.0]


def test_identical_gpus_fill_round_robin():
    """K identical GPUs and identical requests without deadlines: all energies are equal, the tie-breaker
    takes the most free memory, and the commit lowers it by Req_mem: the requests go round robin."""
    K, n = 7, 5
    lat, pw, models, st, rq = _toy(K=K, F=2)
    for k in range(K):
        _gpu(st, k, 1, 2, 1, 0.0, 1e5)
    rq = np.repeat(rq, n * K); rq["slo_ttft_ms"] = 1e9; rq["o_pred"] = 3
    got, after = oracle.dispatch_commit(lat, pw, models, st, rq)
    assert got["gpu"].tolist() == list(range(K)) * n
    assert np.all(after["mem_free_mb"] == f32(1e5) - n * 5.0) and np.all(after["f_cur"] == 1)
    # every request: prefill 1 ms + 4 decode rounds of 1 ms after the previous one on the same GPU
    assert np.all(after["t_avail_ms"] == n * 5.0)
    assert got["ttft_ms"].reshape(n, K)[:, 0].tolist() == [1.0 + 5.0 * i for i in range(n)]


def _variant(seed):
    cl = synth.make_custom(seed=1200 + seed, K=[3, 6, 11][seed % 3], M=3, F=5, S=[4, 8][seed % 2], B=6, R=40, lo=1, hi=4)
    if seed % 4 == 1:
        cl.requests["slo_ttft_ms"] *= 0.05                 # phases 2 and 3 appear as the queues grow
    if seed % 4 == 2:
        cl.states["mem_free_mb"] *= 0.02                   # memory runs out during the batch
    return cl


@pytest.mark.parametrize("seed", range(24))
def test_commit_replayed_with_the_independent_restatement(seed):
    """Each decision equals the independent Python restatement of the three phases (test_oracle_dispatch)
    on the records as they stand before the request, and each commit equals the reading's three updates."""
    cl = _variant(seed)
    got, after = oracle.dispatch_commit(cl.lat, cl.pow, cl.models, cl.states, cl.requests)
    st = cl.states.copy()
    cur = types.SimpleNamespace(**{k: getattr(cl, k) for k in ("lat", "pow", "models", "requests", "K", "F", "S", "B")})
    cur.states = st
    for r in range(cl.R):
        k, sg, phi, phase, e = _restate(cur, r)
        o = got[r]
        assert (int(o["gpu"]), int(o["sigma"]), int(o["phi"]), int(o["f_req"])) == (k, sg, phi, phase), (seed, r)
        if k < 0:
            continue
        rq = cl.requests[r]; m = int(rq["model"]); L = int(rq["L"]); O = (21 * int(rq["o_pred"]) + 19) // 20
        g = st[k]
        js = [i for i in range(int(g["n_res"])) if int(g["t"][i]["model"]) == m]
        wait = g["t_avail_ms"] if js else f32(g["t_avail_ms"] + cl.models["load_ms"][m])
        br1 = int(g["t"][js[0]]["beta"][1]) + 1 if (js and g["t"][js[0]]["q"][1] > 0) else 0
        br0 = max(min(L, cl.B) - 1, 0)
        t0 = f32(f32(-(-L // (br0 + 1))) * cl.lat[m, 0, phi, sg, br0]) if L else f32(0)
        t1 = f32(f32(-(-O // (br1 + 1))) * cl.lat[m, 1, phi, sg, br1]) if O else f32(0)
        st["t_avail_ms"][k] = f32(f32(wait + t0) + t1)
        st["mem_free_mb"][k] = f32(g["mem_free_mb"] - f32(f32(L + O) * cl.models["kv_mb_per_token"][m]))
        st["f_cur"][k] = phi
    assert st.tobytes() == after.tobytes()


def test_commit_invariants_and_difference_from_the_snapshot():
    differs = 0
    for seed in range(24):
        cl = _variant(seed)
        got, after = oracle.dispatch_commit(cl.lat, cl.pow, cl.models, cl.states, cl.requests)
        snap = oracle.dispatch(cl.lat, cl.pow, cl.models, cl.states, cl.requests)
        assert got[0].tobytes() == snap[0].tobytes()         # the first request sees the polled records
        differs += int((got["gpu"] != snap["gpu"]).any())
        assert np.all(after["t_avail_ms"] >= cl.states["t_avail_ms"])
        assert np.all(after["mem_free_mb"] <= cl.states["mem_free_mb"]) and np.all(after["mem_free_mb"] >= 0)
        placed = got["gpu"] >= 0
        untouched = np.setdiff1d(np.arange(cl.K), got["gpu"][placed])
        assert after[untouched].tobytes() == cl.states[untouched].tobytes()
        # tenants, n_res: never touched (the resident set is the last poll's)
        assert after["t"].tobytes() == cl.states["t"].tobytes() and np.array_equal(after["n_res"], cl.states["n_res"])
        # a batch in which everything scales out leaves the records as they were
        cl.states["mem_free_mb"] = 0.5
        got, after = oracle.dispatch_commit(cl.lat, cl.pow, cl.models, cl.states, cl.requests)
        assert np.all(got["gpu"] == -1) and after.tobytes() == cl.states.tobytes()
    assert differs >= 12                                      # the commit pass matters on these inputs
