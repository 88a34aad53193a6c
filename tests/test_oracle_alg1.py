"""Pins of the oracle's Algorithm 1 phase 1 (per-LLM preferred configuration, Eq. 8, Little's law:
PAPER.md lines 277, 337-339) and of the Energy Waste Ratio (Eq. 5-7).  CPU only."""
from __future__ import annotations

import numpy as np
import pytest

import oracle
from paper_2606_30391_b200 import synth

f32 = np.float32


def test_eq8_and_littles_law_by_hand():
    """F = 2, S = 4, one model.  Prefill is cheapest at (phi 1, 4 units): T_p = 100 ms; decode at
    (phi 0, 2 units): T_d = 300 ms  ->  SM_l = (4*100 + 2*300) / 400 = 2.5 units (Eq. 8) -> l.S = 3."""
    M, F, S, B = 1, 2, 4, 4
    lat = np.full((M, 2, F, S, B), 1000.0, dtype=f32); pw = np.full_like(lat, 100.0)
    L, O = 8, 100                                           # prefill bucket min(L,B)-1 = 3, rounds = 2
    lat[0, 0, 1, 3, 3] = 50.0; pw[0, 0, 1, 3, 3] = 10.0     # T_p = 2*50 = 100, e = 1000
    lat[0, 1, 0, 1, 0] = 3.0; pw[0, 1, 0, 1, 0] = 10.0      # T_d = 100*3 = 300, e = 3000
    # at l.S = 3 units (sigma 2): phi 0 -> prefill 2*200*10 = 4000, decode 100*4*10 = 4000 (total 8000);
    #                             phi 1 -> prefill 2*100*10 = 2000, decode 100*5*10 = 5000 (total 7000) -> F_l = 1
    lat[0, 0, 0, 2, 3] = 200.0; pw[0, 0, 0, 2, 3] = 10.0; lat[0, 1, 0, 2, 0] = 4.0; pw[0, 1, 0, 2, 0] = 10.0
    lat[0, 0, 1, 2, 3] = 100.0; pw[0, 0, 1, 2, 3] = 10.0; lat[0, 1, 1, 2, 0] = 5.0; pw[0, 1, 1, 2, 0] = 10.0
    models = np.zeros(1, dtype=synth.MODEL_INFO_DT); models["kv_mb_per_token"] = 0.5; models["weights_mb"] = 14000.0
    llm = np.zeros(1, dtype=synth.LLM_DT)
    llm["avg_in"] = L; llm["avg_out"] = O; llm["slo_ttft_ms"] = 1e9; llm["slo_tbt_ms"] = 1e9; llm["lambda_rps"] = 2.0
    o = oracle.llm_profile(lat, pw, models, llm)[0]
    assert (o["sigma_p"], o["phi_p"], o["sigma_d"], o["phi_d"]) == (3, 1, 1, 0)
    assert (o["t_p_ms"], o["t_d_ms"], o["p_p_w"], o["p_d_w"]) == (100.0, 300.0, 10.0, 10.0)
    assert o["sm_units"] == f32(2.5) and o["need_units"] == 3
    assert o["phi_l"] == 1 and o["e_l_mj"] == f32(7000.0) and o["t_l_ms"] == f32(700.0)
    # Little's law: N_conc = lambda * W = 2 req/s * 0.7 s = 1.4; KV per sequence = 108 tokens * 0.5 MB = 54 MB
    assert o["mem_mb"] == f32(f32(14000.0) + f32(f32(2.0) * f32(f32(700.0) / f32(1000.0))) * f32(54.0))
    assert abs(float(o["mem_mb"]) - (14000.0 + 1.4 * 54.0)) < 1e-2
    # a TBT SLO of 3.5 ms rules out every decode entry but the 3 ms one; F_l then has no feasible frequency at 3 units
    llm["slo_tbt_ms"] = 3.5
    o = oracle.llm_profile(lat, pw, models, llm)[0]
    assert (o["sigma_d"], o["phi_d"], o["need_units"], o["phi_l"]) == (1, 0, 3, -1) and np.isinf(o["mem_mb"])
    llm["slo_tbt_ms"] = 1.0                                  # decode infeasible everywhere
    o = oracle.llm_profile(lat, pw, models, llm)[0]
    assert o["phi_d"] == -1 and o["need_units"] == -1


def _restate(cl, l):
    m, L, O = int(l["model"]), int(l["avg_in"]), int(l["avg_out"])
    b0 = max(min(L, cl.B) - 1, 0); r0 = -(-L // (b0 + 1))
    l0, p0 = cl.lat[m, 0, :, :, b0], cl.pow[m, 0, :, :, b0]
    l1, p1 = cl.lat[m, 1, :, :, 0], cl.pow[m, 1, :, :, 0]
    tp = (f32(r0) * l0).astype(f32) if L else np.zeros_like(l0); ep = (tp * p0).astype(f32) if L else np.zeros_like(l0)
    td = (f32(O) * l1).astype(f32) if O else np.zeros_like(l1); ed = (td * p1).astype(f32) if O else np.zeros_like(l1)
    okp = (tp <= l["slo_ttft_ms"]) if L else np.ones(l0.shape, bool)
    okd = (l1 <= l["slo_tbt_ms"]) if O else np.ones(l1.shape, bool)
    if not okp.any() or not okd.any():
        return None
    ip = int(np.argmin(np.where(okp, ep, np.inf))); idd = int(np.argmin(np.where(okd, ed, np.inf)))
    phi_p, sg_p = divmod(ip, cl.S); phi_d, sg_d = divmod(idd, cl.S)
    Tp, Td = tp[phi_p, sg_p], td[phi_d, sg_d]
    tsum = f32(Tp + Td)
    sm = f32(f32(f32(f32(sg_p + 1) * Tp) + f32(f32(sg_d + 1) * Td)) / tsum) if tsum > 0 else f32(1.0)
    need = min(max(int(np.ceil(sm)), 1), cl.S)
    both = okp[:, need - 1] & okd[:, need - 1]
    e = (ep[:, need - 1] + ed[:, need - 1]).astype(f32)
    phi_l = int(np.argmin(np.where(both, e, np.inf))) if both.any() else -1
    return (sg_p, phi_p, sg_d, phi_d, sm, need, phi_l, e[phi_l] if phi_l >= 0 else np.inf)


@pytest.mark.parametrize("seed", range(12))
def test_llm_profile_equals_independent_restatement(seed):
    cl = synth.make_custom(seed=1100 + seed, K=1, M=4, F=[5, 9, 16][seed % 3], S=[4, 8, 10][seed % 3], B=[6, 16][seed % 2], R=0)
    llms = synth.make_llms(seed, 40, cl.M)
    if seed % 4 == 1:
        llms["slo_ttft_ms"] *= 0.02; llms["slo_tbt_ms"] *= 0.2
    if seed % 4 == 2:
        llms["avg_in"][::3] = 0; llms["avg_out"][1::3] = 0
    got = oracle.llm_profile(cl.lat, cl.pow, cl.models, llms)
    for i in range(len(llms)):
        ref = _restate(cl, llms[i]); o = got[i]
        if ref is None:
            assert o["need_units"] == -1 and (o["phi_p"] == -1 or o["phi_d"] == -1)
            continue
        assert (o["sigma_p"], o["phi_p"], o["sigma_d"], o["phi_d"]) == ref[:4], (seed, i)
        assert o["sm_units"] == ref[4] and o["need_units"] == ref[5] and o["phi_l"] == ref[6]
        assert o["e_l_mj"] == ref[7] or (np.isinf(o["e_l_mj"]) and np.isinf(ref[7]))


def test_ewr_closed_forms():
    """Eq. 5-7: EWR = 0 iff every LLM runs at its GPU's frequency; a two-GPU case by hand."""
    fg, w, o, r = oracle.ewr([0, 0, 1, 1], [1200, 1200, 900, 900], [5, 7, 1, 2], 2)
    assert (w, r) == (0.0, 0.0) and list(fg) == [1200.0, 900.0]
    fg, w, o, r = oracle.ewr([0, 0, 1, -1], [1000, 1500, 1200, 900], [1, 2, 3, 4], 2)
    assert list(fg) == [1500.0, 1200.0]
    assert w == 1 * (1500.0 ** 3 - 1000.0 ** 3) and o == 1000.0 ** 3 + 2 * 1500.0 ** 3 + 3 * 1200.0 ** 3
    assert r == w / o
    # moving the 1000 MHz LLM next to the 1200 MHz one lowers the waste (frequency alignment)
    _, w2, _, r2 = oracle.ewr([1, 0, 1, -1], [1000, 1500, 1200, 900], [1, 2, 3, 4], 2)
    assert w2 == 1200.0 ** 3 - 1000.0 ** 3 and r2 < r
    # scaling every execution time leaves the ratio unchanged
    _, _, _, r3 = oracle.ewr([0, 0, 1, -1], [1000, 1500, 1200, 900], [8, 16, 24, 32], 2)
    assert abs(r3 - r) < 1e-15
    assert oracle.ewr([], [], [], 3)[1:] == (0.0, 0.0, 0.0)


def test_ewr_against_numpy():
    st = synth.Stream(5, "ewr")
    n, K = 5000, 300
    g = st.randint(n, -1, K - 1).astype(np.int32); f = st.urange(n, 210, 1980).astype(f32); t = st.urange(n, 1, 1e4).astype(f32)
    fg, w, o, r = oracle.ewr(g, f, t, K)
    ref_fg = np.zeros(K); m = g >= 0
    np.maximum.at(ref_fg, g[m], f[m].astype(np.float64))
    assert np.array_equal(fg, ref_fg.astype(f32))
    F = ref_fg[g[m]]; fl = f[m].astype(np.float64); tt = t[m].astype(np.float64)
    assert abs(w - (tt * (F ** 3 - fl ** 3)).sum()) <= 1e-12 * abs(w)
    assert abs(o - (tt * fl ** 3).sum()) <= 1e-12 * abs(o)
