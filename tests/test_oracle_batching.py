"""Pins of the oracle's local-scheduler steps 1-2 (unified priority score, Eq. 4, PAPER.md lines
241-246; priority-based task batching with bypass, lines 248-250 and the worked table of Fig. 8,
lines 199-205).  CPU only."""
from __future__ import annotations

import numpy as np
import pytest

import oracle
from paper_2606_30391_b200 import synth

f32 = np.float32


def _fig8_cluster(mem_free):
    """One GPU, S = 10 share units (10 % each), one frequency; the six tasks of Fig. 8 in the
    scrambled order P1, P2, P3, D1, D2, D3, each with its own batch bucket so that the LUT can give
    every task the latency that reproduces the printed score."""
    M, F, S, B = 1, 1, 10, 6
    lat = np.ones((M, 2, F, S, B), dtype=f32)
    pw = np.ones_like(lat)
    # name: (phase, SM %, mem MB, printed score, slack, age)
    fig = {"P1": (0, 50, 800, 2.4, 1000.0, 500.0), "P2": (0, 70, 1400, 2.0, 900.0, 400.0),
           "P3": (0, 40, 500, 2.1, 2000.0, 1000.0), "D1": (1, 20, 400, 3.8, 10.0, 7.0),
           "D2": (1, 20, 650, 2.8, 10.0, 9.0), "D3": (1, 20, 500, 3.0, 10.0, 0.0)}
    names = ["P1", "P2", "P3", "D1", "D2", "D3"]
    tasks = np.zeros(6, dtype=synth.TASK_DT)
    for i, nm in enumerate(names):
        ph, sm, mem, score, slack, age = fig[nm]
        denom = slack - age if ph == 0 else slack          # Eq. 4: beta = 1 prefill, 0 decode
        tasks[i] = (0, ph, sm // 10 - 1, i, (0, 0, 0), slack, age, mem, i)
        lat[0, ph, 0, sm // 10 - 1, i] = f32(score * denom)
    st = np.zeros(1, dtype=synth.GPU_STATE_DT)
    st["n_res"] = 1; st["f_cur"] = 0; st["mem_free_mb"] = mem_free
    return lat, pw, st, tasks, names, fig


def test_fig8_steps_1_and_2_worked_table():
    lat, pw, st, tasks, names, fig = _fig8_cluster(mem_free=1e6)
    out = oracle.batch_tasks(lat, pw, st, [0, 6], tasks)
    for i, nm in enumerate(names):                          # the printed scores
        assert out["score"][i] == f32(fig[nm][3]), nm
    order = [names[i] for i in np.argsort(out["rank"])]
    assert order == ["D1", "D3", "D2", "P1", "P3", "P2"]    # "Sort by (priority) Score"
    adm = {nm: int(out["admitted"][i]) for i, nm in enumerate(names)}
    # 60 % of the SMs are taken by the three decodes; P1 (50 %) does not fit the remaining 40 % and
    # is bypassed, P3 (40 %) fits exactly (100 % counts as feasible, reading s7), P2 (70 %) does not
    assert adm == {"D1": 1, "D3": 1, "D2": 1, "P1": 0, "P3": 1, "P2": 0}


def test_fig8_memory_can_be_the_binding_budget():
    lat, pw, st, tasks, names, _ = _fig8_cluster(mem_free=1600.0)   # D1+D3+D2 = 1550 MB
    out = oracle.batch_tasks(lat, pw, st, [0, 6], tasks)
    adm = {nm: int(out["admitted"][i]) for i, nm in enumerate(names)}
    assert adm == {"D1": 1, "D3": 1, "D2": 1, "P1": 0, "P3": 0, "P2": 0}
    st["mem_free_mb"] = 1549.0                               # D2 no longer fits, P3 (500) neither
    out = oracle.batch_tasks(lat, pw, st, [0, 6], tasks)
    adm = {nm: int(out["admitted"][i]) for i, nm in enumerate(names)}
    assert adm == {"D1": 1, "D3": 1, "D2": 0, "P1": 0, "P3": 1, "P2": 0}   # 900 + 500 = 1400, 80 % SMs


def _restate(cl, off, tasks, ids=None):
    """Independent numpy restatement: stable argsort on -score, then a plain greedy walk."""
    out = np.zeros(len(tasks), dtype=synth.TASK_OUT_DT)
    for gi in range(len(off) - 1):
        g = cl.states[gi if ids is None else ids[gi]]
        t = tasks[off[gi]:off[gi + 1]]
        lat = cl.lat[t["model"], t["phase"], int(g["f_cur"]), t["sigma"], t["beta"]].astype(f32)
        denom = np.where(t["phase"] == 0, (t["slack_ms"] - t["age_ms"]).astype(f32), t["slack_ms"])
        with np.errstate(divide="ignore", invalid="ignore"):
            score = np.where(denom > 0, (lat / denom.astype(f32)).astype(f32), f32(np.inf))
        order = np.argsort(-score.astype(np.float64), kind="stable")
        sm, mem = cl.S, f32(g["mem_free_mb"])
        o = out[off[gi]:off[gi + 1]]
        o["score"] = score; o["latency_ms"] = lat
        for pos, i in enumerate(order):
            o["rank"][i] = pos
            need = int(t["sigma"][i]) + 1
            if need <= sm and t["mem_mb"][i] <= mem:
                o["admitted"][i] = 1; sm -= need; mem = f32(mem - t["mem_mb"][i])
    return out


@pytest.mark.parametrize("seed", range(20))
def test_batching_equals_independent_restatement(seed):
    cl = synth.make_custom(seed=700 + seed, K=7, M=3, F=5, S=[4, 8, 10, 16][seed % 4], B=6, R=0)
    off, tasks = synth.make_tasks(seed, cl.K, cl.M, cl.S, cl.B, 0, 40)
    if seed % 3 == 0:                                        # exact score ties: lowest index first
        tasks["slack_ms"] = 100.0; tasks["age_ms"] = 0.0; tasks["beta"] = 0; tasks["sigma"] = tasks["sigma"] % 2
        tasks["model"] = 0
    got = oracle.batch_tasks(cl.lat, cl.pow, cl.states, off, tasks)
    ref = _restate(cl, off, tasks)
    for f in ("rank", "admitted"):
        assert np.array_equal(got[f], ref[f]), f
    for f in ("score", "latency_ms"):
        assert np.array_equal(got[f].view(np.uint32), ref[f].view(np.uint32)), f


def test_batching_invariants():
    cl = synth.make_custom(seed=77, K=16, M=4, F=8, S=16, B=8, R=0)
    off, tasks = synth.make_tasks(3, cl.K, cl.M, cl.S, cl.B, 10, 100)
    out = oracle.batch_tasks(cl.lat, cl.pow, cl.states, off, tasks)
    for g in range(cl.K):
        t, o = tasks[off[g]:off[g + 1]], out[off[g]:off[g + 1]]
        order = np.argsort(o["rank"])
        assert sorted(o["rank"]) == list(range(len(t)))
        sc = o["score"][order]
        assert (sc[:-1] >= sc[1:]).all()                     # descending score
        adm = o["admitted"] == 1
        assert (t["sigma"][adm].astype(int) + 1).sum() <= cl.S
        assert t["mem_mb"][adm].astype(np.float64).sum() <= float(cl.states["mem_free_mb"][g]) * (1 + 1e-6)
        # a bypassed task did not fit what was left at its turn
        sm, mem = cl.S, float(cl.states["mem_free_mb"][g])
        for i in order:
            need = int(t["sigma"][i]) + 1
            if adm[i]:
                sm -= need; mem = float(f32(f32(mem) - t["mem_mb"][i]))
            else:
                assert need > sm or t["mem_mb"][i] > f32(mem)
        # slack used up (prefill waited longer than its slack) -> most urgent
        gone = (t["phase"] == 0) & (t["slack_ms"] - t["age_ms"] <= 0)
        assert np.isinf(o["score"][gone]).all()


def test_eq4_age_only_counts_for_prefill():
    cl = synth.make_custom(seed=78, K=1, M=2, F=4, S=8, B=4, R=0)
    off, tasks = synth.make_tasks(5, 1, cl.M, cl.S, cl.B, 30, 30)
    tasks["slack_ms"] = 500.0; tasks["age_ms"] = 10.0
    a = oracle.batch_tasks(cl.lat, cl.pow, cl.states, off, tasks)
    tasks["age_ms"] = 300.0
    b = oracle.batch_tasks(cl.lat, cl.pow, cl.states, off, tasks)
    dec, pre = tasks["phase"] == 1, tasks["phase"] == 0
    assert np.array_equal(a["score"][dec], b["score"][dec])            # beta = 0
    assert (b["score"][pre] > a["score"][pre]).all()                   # beta = 1: waiting raises urgency
    assert np.array_equal(a["score"][dec], (a["latency_ms"][dec] / f32(500.0)).astype(f32))
    assert np.array_equal(b["score"][pre], (b["latency_ms"][pre] / f32(200.0)).astype(f32))
