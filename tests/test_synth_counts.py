"""bench_work.eligible_work (the size of the dense definition's candidate set, used by bench.py for its rates)
against a plain double loop over (request, GPU), and the workload variants' shapes."""
from __future__ import annotations

import numpy as np
import pytest

from paper_2606_30391_b200 import synth
import bench_work

f32 = np.float32


def _loop_count(cl):
    pairs = cands = 0
    for rq in cl.requests:
        m = int(rq["model"])
        O = (21 * int(rq["o_pred"]) + 19) // 20
        mem = f32(f32(int(rq["L"]) + O) * cl.models["kv_mb_per_token"][m])
        for g in cl.states:
            n = int(g["n_res"])
            if n < 1 or not (mem <= g["mem_free_mb"]):
                continue
            smf = cl.S - sum(int(g["t"][i]["sigma"]) + 1 for i in range(n))
            if smf < 1:
                continue
            js = [i for i in range(n) if int(g["t"][i]["model"]) == m]
            if js:
                t = g["t"][js[0]]
                if (int(t["beta"][1]) + 1 if t["q"][1] > 0 else 0) >= cl.B:
                    continue
            elif n >= 4:
                continue
            pairs += 1
            cands += smf * cl.F
    return pairs, cands


@pytest.mark.parametrize("seed", range(4))
def test_eligible_work_equals_double_loop(seed):
    cl = synth.make_custom(seed=900 + seed, K=23, M=3, F=5, S=6, B=4, R=57, lo=1, hi=4)
    cl.states["mem_free_mb"][::3] *= 0.05                     # some GPUs too full for most requests
    cl.states["n_res"][1] = 0
    assert bench_work.eligible_work(cl) == _loop_count(cl)


def test_variants_keep_the_shape_and_change_what_they_say():
    base = synth.make_cluster("tiny")
    for v in bench_work.VARIANTS:
        cl = bench_work.make_variant("tiny", v)
        assert cl.lat.shape == base.lat.shape and cl.K == base.K and cl.R == base.R
    assert np.all(bench_work.make_variant("tiny", "dynamic_power_x4").pow >= base.pow)
    assert np.all(bench_work.make_variant("tiny", "cold_starts_feasible").models["load_ms"] < base.models["load_ms"])
    t = bench_work.make_variant("tiny", "ties")
    assert len(np.unique(t.lat)) <= 3 and len(np.unique(t.pow)) <= 2
    with pytest.raises(ValueError):
        bench_work.make_variant("tiny", "nope")
