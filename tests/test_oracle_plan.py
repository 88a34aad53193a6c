"""Pins of the oracle's Algorithm 1 phases 2-3 (PAPER.md lines 282-332 and the prose of lines 341-357):
Best-Fit-Decreasing capacity planning and the EWR-minimising placement loop.  CPU only."""
from __future__ import annotations

import itertools

import numpy as np
import pytest

import oracle
from paper_2606_30391_b200 import synth


def _llms(units, mem, f, t=None):
    n = len(units)
    l = np.zeros(n, dtype=synth.PLAN_LLM_DT)
    l["need_units"] = units; l["mem_mb"] = mem; l["f_mhz"] = f; l["t_ms"] = np.ones(n) if t is None else t
    return l


def _opt_bins(sizes, cap):
    """Optimal bin count by brute force over assignments (tiny n)."""
    n = len(sizes)
    for k in range(1, n + 1):
        for assign in itertools.product(range(k), repeat=n):
            load = [0.0] * k
            for s, b in zip(sizes, assign):
                load[b] += s
            if max(load) <= cap:
                return k
    return n


def test_bfd_by_hand():
    # sizes 7 5 4 3 3 2, capacity 10: 7|3, 5+4, 3+2 ... best fit puts the first 3 beside the 7 -> 3 bins (= optimum)
    l = _llms([7, 5, 4, 3, 3, 2], [1.0] * 6, [1000] * 6)
    _, (n_sm, n_mem, n_min, _) = oracle.replace_plan(l, 10, 1e6)
    assert (n_sm, n_mem, n_min) == (3, 1, 3)
    # the same sizes as memory
    l = _llms([1] * 6, [7, 5, 4, 3, 3, 2], [1000] * 6)
    _, (n_sm, n_mem, n_min, _) = oracle.replace_plan(l, 100, 10.0)
    assert (n_sm, n_mem, n_min) == (1, 3, 3)
    # first-fit-decreasing would need 3 bins here too, but best fit must pick the FULLEST bin that fits:
    # 6 5 | 4 -> beside the 6 (room 4), not the 5 (room 5); then 5 beside the 5: 2 bins
    l = _llms([6, 5, 4, 5], [1.0] * 4, [1000] * 4)
    assert oracle.replace_plan(l, 10, 1e6)[1][0] == 2


@pytest.mark.parametrize("seed", range(25))
def test_bfd_against_brute_force_optimum(seed):
    st = synth.Stream(seed, "bfd")
    n = int(st.randint(1, 1, 7)[0]); cap = int(st.randint(1, 6, 16)[0])
    units = st.randint(n, 1, cap).astype(int)
    l = _llms(units, [1.0] * n, [1000] * n)
    n_sm = oracle.replace_plan(l, cap, 1e6)[1][0]
    opt = _opt_bins(list(units), cap)
    assert opt <= n_sm <= (11 * opt) // 9 + 1                # the classical BFD guarantee
    mem = (st.urange(n, 0.05, 1.0) * 100).astype(np.float32)
    l = _llms([1] * n, mem, [1000] * n)
    n_mem = oracle.replace_plan(l, 1000, 100.0)[1][1]
    opt = _opt_bins([float(x) for x in mem], 100.0)
    assert opt <= n_mem <= (11 * opt) // 9 + 1


def test_fig9_direct_placement_then_ewr_driven_swap():
    """Fig. 9: LLMs are placed by ascending preferred frequency next to the closest
    GPU frequency; when the target lacks memory for the newcomer, the resident with the LOWEST frequency
    (the outlier) moves to the candidate GPU if that is resource-valid and lowers the waste."""
    #            A     B     C     D (newcomer, highest F)
    l = _llms([1, 1, 1, 1], [30, 30, 30, 40], [900, 1000, 1400, 1500], [10, 10, 10, 10])
    gpu_of, (n_sm, n_mem, n_min, n_act) = oracle.replace_plan(l, 10, 100.0)
    assert (n_mem, n_min, n_act) == (2, 2, 2)
    # A, B, C group on GPU 0 (direct placement: 90 of 100 MB); D (40 MB) does not fit; A (900 MHz) is the
    # outlier: GPU 1 can take it, GPU 0 without A has 40 MB free, and the waste drops by t_A (1500^3 - 900^3)
    assert list(gpu_of) == [1, 0, 0, 0]
    before = oracle.ewr([0, 0, 0, 0], l["f_mhz"], l["t_ms"], 2)[1]
    after = oracle.ewr(gpu_of, l["f_mhz"], l["t_ms"], 2)[1]
    assert before - after == 10 * (1500.0 ** 3 - 900.0 ** 3)
    # if the outlier's departure does not free enough memory, no swap: the newcomer goes to the candidate GPU
    l["mem_mb"][3] = 50
    assert list(oracle.replace_plan(l, 10, 100.0)[0]) == [0, 0, 0, 1]
    # if nothing fits anywhere, a new GPU is activated (Alg. 1 l.26-27)
    l = _llms([1, 1, 1], [60, 60, 60], [900, 1000, 1100])
    gpu_of, summ = oracle.replace_plan(l, 10, 100.0)
    assert sorted(gpu_of) == [0, 1, 2] and summ[3] == 3
    # an LLM that exceeds a whole GPU stays unplaced
    l = _llms([11, 1], [10, 10], [900, 1000])
    assert list(oracle.replace_plan(l, 10, 100.0)[0]) == [-1, 0]


@pytest.mark.parametrize("seed", range(10))
def test_plan_invariants(seed):
    freq = np.linspace(210, 1980, 32).astype(np.float32)
    S_eff, M_eff = 15, 76000.0
    l = synth.make_plan_llms(seed, 40 + 30 * seed, 16, freq)
    gpu_of, (n_sm, n_mem, n_min, n_act) = oracle.replace_plan(l, S_eff, M_eff)
    assert (gpu_of >= 0).all() and gpu_of.max() == n_act - 1 and n_act >= n_min == max(n_sm, n_mem)
    assert n_sm >= -(-int(l["need_units"].sum()) // S_eff) and n_mem >= int(np.ceil(l["mem_mb"].astype(np.float64).sum() / M_eff))
    for g in range(n_act):
        m = gpu_of == g
        assert l["need_units"][m].sum() <= S_eff and l["mem_mb"][m].astype(np.float64).sum() <= M_eff * (1 + 1e-6)
    # grouping by frequency beats spreading the same LLMs round-robin over the same number of GPUs
    ewr_plan = oracle.ewr(gpu_of, l["f_mhz"], l["t_ms"], n_act)[3]
    ewr_rr = oracle.ewr(np.arange(len(l)) % n_act, l["f_mhz"], l["t_ms"], n_act)[3]
    assert ewr_plan < 0.5 * ewr_rr
