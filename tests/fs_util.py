"""Hand-built inputs for the pins (tests only)."""
from __future__ import annotations

import numpy as np

from paper_2606_30391_b200 import synth


def mk_state(f_cur=0, t_avail=0.0, mem_free=1e6, tenants=()):
    g = np.zeros((), dtype=synth.GPU_STATE_DT)
    g["n_res"] = len(tenants)
    g["f_cur"] = f_cur
    g["t_avail_ms"] = t_avail
    g["mem_free_mb"] = mem_free
    for i, t in enumerate(tenants):
        g["t"][i]["model"] = t.get("model", 0)
        g["t"][i]["sigma"] = t.get("sigma", 0)
        g["t"][i]["beta"] = t.get("beta", (0, 0))
        g["t"][i]["q"] = t.get("q", (0, 0))
        g["t"][i]["slo_ms"] = t.get("slo", (1e9, 1e9))
        g["t"][i]["mem_used_mb"] = t.get("mem", 0.0)
    return g


def mk_states(lst):
    return np.array(lst, dtype=synth.GPU_STATE_DT)


def mk_requests(lst):
    r = np.zeros(len(lst), dtype=synth.REQUEST_DT)
    for i, d in enumerate(lst):
        r[i]["model"] = d.get("model", 0)
        r[i]["L"] = d.get("L", 1)
        r[i]["o_pred"] = d.get("o_pred", 0)
        r[i]["slo_ttft_ms"] = d.get("ttft", 1e9)
        r[i]["slo_tbt_ms"] = d.get("tbt", 1e9)
        r[i]["tag"] = i
    return r


def mk_models(M, load_ms=0.0, kv=0.0, weights=0.0, mig=0.0):
    m = np.zeros(M, dtype=synth.MODEL_INFO_DT)
    m["load_ms"] = load_ms
    m["kv_mb_per_token"] = kv
    m["weights_mb"] = weights
    m["mig_mj"] = mig
    return m


def cluster_from(lat, pow_, models, states, requests, params=None):
    M, _, F, S, B = lat.shape
    return synth.Cluster(name="hand", M=M, F=F, S=S, B=B, K=len(states),
                         lat=np.ascontiguousarray(lat, dtype=np.float32),
                         pow=np.ascontiguousarray(pow_, dtype=np.float32),
                         freq_mhz=np.arange(F, dtype=np.float32), models=models, states=states,
                         requests=requests, params=params or synth.Params())


def tie_heavy(cl, seed):
    """Quantise the tables to a few power-of-two values so that exact ties abound."""
    st = synth.Stream(seed, "ties")
    n = cl.lat.size
    cl.lat[...] = (2.0 ** st.randint(n, 0, 2)).reshape(cl.lat.shape).astype(np.float32)
    cl.pow[...] = (64.0 * 2.0 ** st.randint(n, 0, 1)).reshape(cl.pow.shape).astype(np.float32)
    return cl
