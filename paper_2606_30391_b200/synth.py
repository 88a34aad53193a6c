"""Seeded synthetic clusters shaped like the paper's workloads (test / bench infrastructure).

This module is the ONLY code shared by the CPU oracle (`oracle/`) and the CUDA path
(`paper_2606_30391_b200/csrc`).  It holds none of the method's arithmetic: it only draws
profile tables, per-GPU state records and request records, in the byte layout of
`include/festina_eval.h`, from a counter-based generator (SplitMix64).  The recipe is stated in
DESIGN.md ("Input recipe"); it follows BASELINE.json's `configs` (lognormal lengths, SLO ranges,
peak/valley ratios 3.3x and 34.6x from PAPER.md line 40, Beta(2,5) utilisation).  The inputs are
synthetic stand-ins for the paper's ShareGPT / Azure-trace workloads, not reproductions of them.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

RMAX = 4

# ---- record layouts (mirrors of include/festina_eval.h; sizes asserted below) -------------
TENANT_DT = np.dtype(
    [("model", "<i2"), ("sigma", "u1"), ("_p0", "u1"), ("beta", "u1", (2,)), ("_p1", "u1", (2,)),
     ("q", "<u4", (2,)), ("slo_ms", "<f4", (2,)), ("mem_used_mb", "<f4")])
GPU_STATE_DT = np.dtype(
    [("n_res", "<i4"), ("f_cur", "<i4"), ("t_avail_ms", "<f4"), ("mem_free_mb", "<f4"),
     ("t", TENANT_DT, (RMAX,))])
REQUEST_DT = np.dtype(
    [("model", "<i4"), ("L", "<u4"), ("o_pred", "<u4"), ("slo_ttft_ms", "<f4"),
     ("slo_tbt_ms", "<f4"), ("tag", "<u4"), ("_pad", "<u4", (2,))])
MODEL_INFO_DT = np.dtype(
    [("load_ms", "<f4"), ("kv_mb_per_token", "<f4"), ("weights_mb", "<f4"), ("mig_mj", "<f4")])
PLACEMENT_DT = np.dtype(
    [("gpu", "<i4"), ("sigma", "<i2"), ("phi", "<i2"), ("beta", "<i2"), ("f_req", "<i2"),
     ("energy_mj", "<f4"), ("ttft_ms", "<f4"), ("tbt_ms", "<f4"), ("flat", "<u4"), ("_pad", "<u4")])
GPU_AVAIL_DT = np.dtype([("t_avail_ms", "<f4"), ("mem_free_mb", "<f4"), ("f_cur", "<i4"), ("_pad", "<u4")])
LOCAL_CFG_DT = np.dtype(
    [("phi", "<i2"), ("f_req", "<i2"), ("sigma", "u1", (RMAX,)), ("beta", "u1", (RMAX, 2)),
     ("cost", "<f4"), ("energy_mj", "<f4"), ("power_w", "<f4"), ("flat", "<u4"),
     ("_pad", "<u4", (4,))])
CONSOL_DT = np.dtype([("dst", "<i4"), ("phi", "<i4"), ("score_mj", "<f4"), ("saving_mj", "<f4")])
TASK_DT = np.dtype([("model", "<i2"), ("phase", "u1"), ("sigma", "u1"), ("beta", "u1"), ("_p0", "u1", (3,)),
                    ("slack_ms", "<f4"), ("age_ms", "<f4"), ("mem_mb", "<f4"), ("tag", "<u4")])
TASK_OUT_DT = np.dtype([("score", "<f4"), ("latency_ms", "<f4"), ("rank", "<i4"), ("admitted", "<i4")])
LLM_DT = np.dtype([("model", "<i4"), ("avg_in", "<u4"), ("avg_out", "<u4"), ("slo_ttft_ms", "<f4"),
                   ("slo_tbt_ms", "<f4"), ("lambda_rps", "<f4"), ("_pad", "<u4", (2,))])
LLM_PROFILE_DT = np.dtype([("sigma_p", "<i2"), ("phi_p", "<i2"), ("sigma_d", "<i2"), ("phi_d", "<i2"),
                           ("t_p_ms", "<f4"), ("t_d_ms", "<f4"), ("p_p_w", "<f4"), ("p_d_w", "<f4"),
                           ("sm_units", "<f4"), ("need_units", "<i2"), ("phi_l", "<i2"), ("t_l_ms", "<f4"),
                           ("e_l_mj", "<f4"), ("mem_mb", "<f4"), ("_pad", "<u4")])
assert TASK_DT.itemsize == 24 and TASK_OUT_DT.itemsize == 16
MIG_REQ_DT = np.dtype([("remaining_ms", "<f4"), ("tokens_mb", "<f4"), ("kv_mb", "<f4"), ("bw_mb_per_ms", "<f4"),
                       ("recompute_ms", "<f4"), ("_pad", "<u4", (3,))])
assert MIG_REQ_DT.itemsize == 32
PLAN_LLM_DT = np.dtype([("need_units", "<i4"), ("mem_mb", "<f4"), ("f_mhz", "<f4"), ("t_ms", "<f4")])
assert LLM_DT.itemsize == 32 and LLM_PROFILE_DT.itemsize == 48 and PLAN_LLM_DT.itemsize == 16

assert TENANT_DT.itemsize == 28 and GPU_STATE_DT.itemsize == 128 and REQUEST_DT.itemsize == 32
assert MODEL_INFO_DT.itemsize == 16 and PLACEMENT_DT.itemsize == 32
assert LOCAL_CFG_DT.itemsize == 48 and CONSOL_DT.itemsize == 16


@dataclass
class Params:
    p_idle_w: float = 98.7       # derived from PAPER.md line 623 (29.6 kJ per 5 min)
    horizon_ms: float = 300000.0  # Delta = 5 min
    mem_cap_mb: float = 80000.0
    delta_pct: int = 5


@dataclass
class Cluster:
    """One synthetic problem instance: tables + GPU states (+ requests)."""
    name: str
    M: int
    F: int
    S: int
    B: int
    K: int
    lat: np.ndarray            # [M,2,F,S,B] float32 (ms)
    pow: np.ndarray            # [M,2,F,S,B] float32 (W)
    freq_mhz: np.ndarray       # [F] float32
    models: np.ndarray         # [M] MODEL_INFO_DT
    states: np.ndarray         # [K] GPU_STATE_DT
    requests: np.ndarray       # [R] REQUEST_DT
    params: Params = field(default_factory=Params)
    seed: int = 0

    @property
    def R(self) -> int:
        return int(self.requests.shape[0])

    @property
    def dense_candidates(self) -> int:
        """Nominal dense placement grid R*K*S*F."""
        return self.R * self.K * self.S * self.F


# ---- counter-based generator ---------------------------------------------------------------
_GAMMA = np.uint64(0x9E3779B97F4A7C15)
_M1 = np.uint64(0xBF58476D1CE4E5B9)
_M2 = np.uint64(0x94D049BB133111EB)


def _fnv1a(name: str) -> int:
    h = 0xCBF29CE484222325
    for ch in name.encode():
        h = ((h ^ ch) * 0x100000001B3) & 0xFFFFFFFFFFFFFFFF
    return h


class Stream:
    """SplitMix64 stream `seed xor FNV1a(name)`; draws are consumed in order."""

    def __init__(self, seed: int, name: str):
        self.state = np.uint64((seed ^ _fnv1a(name)) & 0xFFFFFFFFFFFFFFFF)

    def u64(self, n: int) -> np.ndarray:
        with np.errstate(over="ignore"):
            idx = np.arange(1, n + 1, dtype=np.uint64)
            z = self.state + idx * _GAMMA
            self.state = self.state + np.uint64(n) * _GAMMA
            z = (z ^ (z >> np.uint64(30))) * _M1
            z = (z ^ (z >> np.uint64(27))) * _M2
            z = z ^ (z >> np.uint64(31))
        return z

    def uniform(self, n: int) -> np.ndarray:
        """U[0,1) with 24 random bits, as float64."""
        return (self.u64(n) >> np.uint64(40)).astype(np.float64) * (2.0 ** -24)

    def urange(self, n: int, lo: float, hi: float) -> np.ndarray:
        return lo + (hi - lo) * self.uniform(n)

    def randint(self, n: int, lo, hi) -> np.ndarray:
        """Integers uniform in [lo, hi] inclusive (lo/hi scalars or arrays of length n)."""
        lo = np.asarray(lo, dtype=np.int64)
        hi = np.asarray(hi, dtype=np.int64)
        span = (hi - lo + 1).astype(np.float64)
        return lo + np.minimum(np.floor(self.uniform(n) * span).astype(np.int64), hi - lo)

    def normal(self, n: int) -> np.ndarray:
        """Box-Muller in double."""
        u1 = 1.0 - self.uniform(n)  # (0,1]
        u2 = self.uniform(n)
        return np.sqrt(-2.0 * np.log(u1)) * np.cos(2.0 * np.pi * u2)

    def lognormal_len(self, n: int, mu: float, sigma: float, cap: int) -> np.ndarray:
        """min(floor(lognormal(mu, sigma)) + 1, cap) as int64 (token counts)."""
        x = np.exp(mu + sigma * self.normal(n))
        return np.minimum(np.floor(x).astype(np.int64) + 1, cap)

    def beta25(self, n: int) -> np.ndarray:
        """Beta(2,5) via order statistics of 6 uniforms (2nd smallest)."""
        u = np.sort(self.uniform(n * 6).reshape(n, 6), axis=1)
        return u[:, 1]


# ---- profile tables ------------------------------------------------------------------------
def table_coeffs(seed: int, M: int):
    """The per-(model, phase) coefficients a, b, c [M,2] and per-model P_s [M] of make_tables."""
    st = Stream(seed, "tables")
    a = st.urange(M * 2, 0.5, 2.0).reshape(M, 2)
    b = st.urange(M * 2, 0.05, 0.3).reshape(M, 2)
    c = st.urange(M * 2, 0.8, 1.2).reshape(M, 2)
    p_s = Stream(seed, "models").urange(M, 60.0, 90.0)
    return a, b, c, p_s


def make_tables(seed: int, M: int, F: int, S: int, B: int):
    """Analytic LUT of BASELINE.json configs[0], with the unit scaling of DESIGN.md (R:s21).

    LAT[m,p,phi,sigma,beta] = tau_p * n^gamma_p * (a/(fh*sh) + b)         [ms]
    POW[m,p,phi,sigma,beta] = P_s + 600 * c * fh^3 * sh * (0.3 + 0.7 n/B)  [W]
    with fh = f_phi/1980, sh = (sigma+1)/S, n = beta+1.
    """
    st = Stream(seed, "tables")
    a = st.urange(M * 2, 0.5, 2.0).reshape(M, 2)
    b = st.urange(M * 2, 0.05, 0.3).reshape(M, 2)
    c = st.urange(M * 2, 0.8, 1.2).reshape(M, 2)
    sm = Stream(seed, "models")
    p_s = sm.urange(M, 60.0, 90.0)
    models = np.zeros(M, dtype=MODEL_INFO_DT)
    models["load_ms"] = sm.urange(M, 500.0, 3000.0).astype(np.float32)
    models["kv_mb_per_token"] = sm.urange(M, 0.1, 0.8).astype(np.float32)
    w = sm.urange(M, 6000.0, 28000.0)
    models["weights_mb"] = w.astype(np.float32)
    models["mig_mj"] = (0.4 * w).astype(np.float32)

    freq = 210.0 + np.arange(F, dtype=np.float64) * (1770.0 / max(F - 1, 1))
    fh = (freq / 1980.0).reshape(1, 1, F, 1, 1)
    sh = ((np.arange(S, dtype=np.float64) + 1.0) / S).reshape(1, 1, 1, S, 1)
    n = (np.arange(B, dtype=np.float64) + 1.0).reshape(1, 1, 1, 1, B)
    tau = np.array([0.1, 1.0]).reshape(1, 2, 1, 1, 1)
    gam = np.array([0.9, 0.7]).reshape(1, 2, 1, 1, 1)
    A = a.reshape(M, 2, 1, 1, 1)
    Bc = b.reshape(M, 2, 1, 1, 1)
    C = c.reshape(M, 2, 1, 1, 1)
    lat = np.empty((M, 2, F, S, B), dtype=np.float32)
    powr = np.empty((M, 2, F, S, B), dtype=np.float32)
    # per-model loop keeps the float64 temporaries small at M=128, B=128
    for m in range(M):
        lat[m] = (tau * n ** gam * (A[m:m + 1] / (fh * sh) + Bc[m:m + 1]))[0].astype(np.float32)
        powr[m] = (p_s[m] + 600.0 * C[m:m + 1] * fh ** 3 * sh * (0.3 + 0.7 * n / B))[0].astype(np.float32)
    return lat, powr, freq.astype(np.float32), models


# ---- load profiles over time (shape of PAPER.md line 40: peak/valley 3.3x and 34.6x) -------
def _load_multiplier(st: Stream, K: int, profile: str) -> np.ndarray:
    """u_k in [1/rho, 1]: lambda(t)/lambda_peak at a uniform random time, per GPU."""
    if profile == "flat":
        return np.ones(K)
    if profile == "diurnal":      # rho = 3.3, cosine day
        rho = 3.3
        t = st.uniform(K)
        lo = 1.0 / rho
        return lo + (1.0 - lo) * 0.5 * (1.0 + np.cos(2.0 * np.pi * t))
    if profile == "bursty":       # rho = 34.6, two-state burst process: 15 % of time in burst
        rho = 34.6
        burst = st.uniform(K) < 0.15
        lvl = st.uniform(K)
        lo = 1.0 / rho
        return np.where(burst, 0.5 + 0.5 * lvl, lo + (0.25 - lo) * lvl)
    if profile == "beta25":       # utilisation ~ Beta(2,5) (BASELINE.json configs[4])
        return np.maximum(st.beta25(K), 1.0 / 64.0)
    raise ValueError(profile)


def _compositions(st: Stream, K: int, total: np.ndarray, parts: np.ndarray) -> np.ndarray:
    """Uniform random composition of total[k] share units into parts[k] >= 1 positive parts.

    Returns [K, RMAX] int64 (zeros beyond parts[k]).  Stars-and-bars: choose parts-1 distinct
    cut points in 1..total-1 by ranking uniform keys.
    """
    smax = int(total.max()) if K else 1
    keys = st.uniform(K * max(smax - 1, 1)).reshape(K, max(smax - 1, 1))
    pos = np.arange(1, max(smax, 2), dtype=np.int64).reshape(1, -1)
    keys = np.where(pos <= (total.reshape(-1, 1) - 1), keys, 2.0)  # invalid positions last
    order = np.argsort(keys, axis=1, kind="stable")
    out = np.zeros((K, RMAX), dtype=np.int64)
    for k in range(K):
        p = int(parts[k])
        cuts = np.sort(order[k, : p - 1] + 1) if p > 1 else np.zeros(0, dtype=np.int64)
        edges = np.concatenate(([0], cuts, [int(total[k])]))
        out[k, :p] = np.diff(edges)
    return out


def make_states(seed: int, K: int, M: int, F: int, S: int, B: int, models: np.ndarray,
                n_res_lo: int, n_res_hi: int, profile: str, local_sweep: bool = False,
                full_split: bool = False) -> np.ndarray:
    st = Stream(seed, "states")
    n_res = st.randint(K, n_res_lo, n_res_hi)
    u = _load_multiplier(st, K, profile)
    # distinct models per GPU: rank uniform keys
    keys = st.uniform(K * M).reshape(K, M)
    mdl = np.argsort(keys, axis=1, kind="stable")[:, :RMAX]
    if mdl.shape[1] < RMAX:       # M < RMAX: slots beyond n_res (<= M) are dead anyway
        mdl = np.concatenate([mdl, np.zeros((K, RMAX - mdl.shape[1]), dtype=mdl.dtype)], axis=1)
    used_lo = n_res
    used = st.randint(K, used_lo, np.maximum(S - 1, used_lo))
    if full_split:
        used = np.full(K, S, dtype=np.int64)
    shares = _compositions(st, K, used, n_res)
    states = np.zeros(K, dtype=GPU_STATE_DT)
    states["n_res"] = n_res
    states["f_cur"] = st.randint(K, F // 4, F - 1)
    states["t_avail_ms"] = st.urange(K, 0.0, 200.0).astype(np.float32)
    states["mem_free_mb"] = st.urange(K, 2000.0, 40000.0).astype(np.float32)
    half = max(B // 2, 1)
    nseq_raw = st.randint(K * RMAX, 0, half).reshape(K, RMAX)
    lens = st.lognormal_len(K * RMAX * half, 5.0, 1.0, 4096).reshape(K, RMAX, half)
    q0_on = st.uniform(K * RMAX).reshape(K, RMAX) < 0.5
    q0_raw = st.randint(K * RMAX, 1, 1024).reshape(K, RMAX)
    slo0 = st.urange(K * RMAX, 500.0, 2000.0).reshape(K, RMAX)
    slo1 = st.urange(K * RMAX, 50.0, 150.0).reshape(K, RMAX)
    qs = st.randint(K * RMAX * 2, 0, 256).reshape(K, RMAX, 2)   # local-sweep queue depths
    bs = st.randint(K * RMAX * 2, 0, B - 1).reshape(K, RMAX, 2)
    kv = models["kv_mb_per_token"].astype(np.float64)
    wmb = models["weights_mb"].astype(np.float64)
    for i in range(RMAX):
        live = i < n_res
        t = states["t"][:, i]
        if local_sweep:
            q0 = qs[:, i, 0]
            q1 = qs[:, i, 1]
            b0 = bs[:, i, 0]
            b1 = bs[:, i, 1]
        else:
            nseq = np.floor(nseq_raw[:, i] * u + 0.5).astype(np.int64)
            mask = np.arange(half).reshape(1, -1) < nseq.reshape(-1, 1)
            q1 = (lens[:, i, :] * mask).sum(axis=1)
            q0 = np.where(q0_on[:, i], np.maximum(np.floor(q0_raw[:, i] * u).astype(np.int64), 1), 0)
            b0 = np.full(K, B - 1, dtype=np.int64)
            b1 = np.maximum(nseq - 1, 0)
        m = mdl[:, i]
        t["model"] = np.where(live, m, 0)
        t["sigma"] = np.where(live, np.maximum(shares[:, i] - 1, 0), 0)
        t["beta"][:, 0] = np.where(live, b0, 0)
        t["beta"][:, 1] = np.where(live, b1, 0)
        t["q"][:, 0] = np.where(live, q0, 0)
        t["q"][:, 1] = np.where(live, q1, 0)
        t["slo_ms"][:, 0] = np.where(live, slo0[:, i], 0).astype(np.float32)
        t["slo_ms"][:, 1] = np.where(live, slo1[:, i], 0).astype(np.float32)
        t["mem_used_mb"] = np.where(live, wmb[m] + kv[m] * (q0 + q1), 0).astype(np.float32)
        states["t"][:, i] = t
    return states


def make_requests(seed: int, R: int, M: int) -> np.ndarray:
    st = Stream(seed, "requests")
    req = np.zeros(R, dtype=REQUEST_DT)
    req["model"] = st.randint(R, 0, M - 1)
    req["L"] = st.lognormal_len(R, 6.0, 1.0, 4096)
    req["o_pred"] = st.lognormal_len(R, 5.0, 1.0, 4096)
    req["slo_ttft_ms"] = st.urange(R, 500.0, 2000.0).astype(np.float32)
    req["slo_tbt_ms"] = st.urange(R, 50.0, 150.0).astype(np.float32)
    req["tag"] = np.arange(R, dtype=np.uint32)
    return req


def make_tasks(seed: int, K: int, M: int, S: int, B: int, lo: int, hi: int):
    """Runnable tasks per GPU for the local scheduler's steps 1-2 (Eq. 4, Fig. 8): `lo..hi`
    tasks per GPU (the paper's Table 3 measures 10-100 queued tasks), ~60 % decode steps with TBT
    slack U[5,150] ms and ~40 % prefill units with TTFT slack U[50,2000] ms and age U[0,1.2*slack)
    (so some prefills have used up their slack), SM demand 1..S/2 units, KV memory lognormal.
    Returns (off [K+1] int32, tasks [off[K]] TASK_DT)."""
    st = Stream(seed, "tasks")
    n = st.randint(K, lo, hi).astype(np.int64)
    off = np.zeros(K + 1, dtype=np.int32)
    off[1:] = np.cumsum(n)
    T = int(off[-1])
    t = np.zeros(T, dtype=TASK_DT)
    t["model"] = st.randint(T, 0, M - 1)
    ph = (st.uniform(T) < 0.6).astype(np.uint8)          # 1 = decode
    t["phase"] = ph
    t["sigma"] = st.randint(T, 0, max(S // 2 - 1, 0))
    t["beta"] = st.randint(T, 0, B - 1)
    slack = np.where(ph == 1, st.urange(T, 5.0, 150.0), st.urange(T, 50.0, 2000.0))
    t["slack_ms"] = slack.astype(np.float32)
    t["age_ms"] = (st.uniform(T) * 1.2 * slack).astype(np.float32)
    t["mem_mb"] = np.minimum(np.exp(5.5 + st.normal(T)), 8000.0).astype(np.float32)
    t["tag"] = np.arange(T, dtype=np.uint32)
    return off, t


def make_llms(seed: int, n: int, M: int) -> np.ndarray:
    """Active LLMs for Algorithm 1 phase 1: average input / output lengths of the last window
    (capped lognormals as for requests), SLOs in the paper's Table 2 ranges, arrival rate U[0.1, 5] req/s."""
    st = Stream(seed, "llms")
    l = np.zeros(n, dtype=LLM_DT)
    l["model"] = st.randint(n, 0, M - 1)
    l["avg_in"] = st.lognormal_len(n, 6.0, 1.0, 4096)
    l["avg_out"] = st.lognormal_len(n, 5.0, 1.0, 4096)
    l["slo_ttft_ms"] = st.urange(n, 250.0, 2000.0).astype(np.float32)
    l["slo_tbt_ms"] = st.urange(n, 50.0, 150.0).astype(np.float32)
    l["lambda_rps"] = st.urange(n, 0.1, 5.0).astype(np.float32)
    return l


def make_plan_llms(seed: int, n: int, S: int, freq_mhz: np.ndarray, mem_cap: float = 80000.0) -> np.ndarray:
    """LLM descriptors (l.S, l.M, l.F) for Algorithm 1 phases 2-3: SM demand 1..S/2 units, memory
    6-40 % of a GPU (3-14 B parameter models plus KV), preferred frequency one of the table's levels."""
    st = Stream(seed, "plan")
    l = np.zeros(n, dtype=PLAN_LLM_DT)
    l["need_units"] = st.randint(n, 1, max(S // 2, 1))
    l["mem_mb"] = (st.urange(n, 0.06, 0.40) * mem_cap).astype(np.float32)
    l["f_mhz"] = np.asarray(freq_mhz, dtype=np.float32)[st.randint(n, 0, len(freq_mhz) - 1)]
    l["t_ms"] = st.urange(n, 50.0, 5000.0).astype(np.float32)
    return l


def make_migration(seed: int, n: int, r: int):
    """State sizes and link bandwidths for the transmission plan (Appendix E): n sources with
    6-60 GB of weights + KV, bandwidth 450 MB/ms inside a node of 8 (NVLink 5 class), 25-50 MB/ms across
    nodes, a source mapped onto itself moves nothing faster (bw = 1e6); and r in-flight requests."""
    st = Stream(seed, "migration")
    bytes_mb = st.urange(n, 6000.0, 60000.0).astype(np.float32)
    node = np.arange(n) // 8
    same = node[:, None] == node[None, :]
    bw = np.where(same, 450.0, st.urange(n * n, 25.0, 50.0).reshape(n, n)).astype(np.float32)
    bw[np.arange(n), np.arange(n)] = 1e6
    q = np.zeros(r, dtype=MIG_REQ_DT)
    q["remaining_ms"] = np.exp(4.0 + 2.0 * st.normal(r)).astype(np.float32)
    q["tokens_mb"] = st.urange(r, 0.001, 0.05).astype(np.float32)
    q["kv_mb"] = st.urange(r, 10.0, 3000.0).astype(np.float32)
    q["bw_mb_per_ms"] = np.where(st.uniform(r) < 0.5, 450.0, 40.0).astype(np.float32)
    q["recompute_ms"] = st.urange(r, 5.0, 400.0).astype(np.float32)
    return bytes_mb, bw, q


def arrival_ticks(seed: int, R: int, n_ticks: int, rho: float = 3.3) -> np.ndarray:
    """Split R requests into dispatch ticks following a Poisson process whose rate follows a
    cosine day with peak/valley = rho (BASELINE.json configs[1]).  Returns tick sizes (sum R)."""
    st = Stream(seed, "arrivals")
    t = (np.arange(n_ticks) + 0.5) / n_ticks
    lo = 1.0 / rho
    rate = lo + (1.0 - lo) * 0.5 * (1.0 + np.cos(2.0 * np.pi * t))
    cdf = np.cumsum(rate) / rate.sum()
    tick = np.searchsorted(cdf, st.uniform(R), side="left")
    return np.bincount(np.minimum(tick, n_ticks - 1), minlength=n_ticks)


# ---- the five configurations of BASELINE.json ------------------------------------------------
CONFIGS = {
    # name: (seed, K, M, F, S, B, n_res_lo, n_res_hi, R, profile, local_sweep)
    "tiny": dict(seed=0, K=8, M=3, F=16, S=8, B=16, lo=1, hi=3, R=256, profile="flat"),
    "rack": dict(seed=1, K=64, M=16, F=32, S=16, B=64, lo=1, hi=4, R=8192, profile="diurnal"),
    "pod": dict(seed=2, K=1024, M=64, F=64, S=16, B=128, lo=1, hi=4, R=65536, profile="bursty"),
    "local": dict(seed=3, K=4096, M=64, F=64, S=16, B=256, lo=2, hi=4, R=0, profile="flat",
                  local_sweep=True),
    "consol": dict(seed=4, K=4096, M=128, F=64, S=16, B=128, lo=1, hi=2, R=0, profile="beta25"),
}


def make_cluster(name: str, **override) -> Cluster:
    """Build one of BASELINE.json's configs ('tiny','rack','pod','local','consol'); any field
    (K, M, F, S, B, R, seed, lo, hi, profile) can be overridden for reduced-size tests."""
    cfg = dict(CONFIGS[name])
    cfg.update(override)
    seed, K, M, F, S, B = (cfg[k] for k in ("seed", "K", "M", "F", "S", "B"))
    lat, powr, freq, models = make_tables(seed, M, F, S, B)
    states = make_states(seed, K, M, F, S, B, models, cfg["lo"], min(cfg["hi"], M),
                         cfg["profile"], cfg.get("local_sweep", False))
    reqs = make_requests(seed, cfg["R"], M)
    return Cluster(name=name, M=M, F=F, S=S, B=B, K=K, lat=lat, pow=powr, freq_mhz=freq,
                   models=models, states=states, requests=reqs, seed=seed)


def make_custom(seed: int, K: int, M: int, F: int, S: int, B: int, R: int, lo: int = 1,
                hi: int = 4, profile: str = "flat", local_sweep: bool = False) -> Cluster:
    """Free-form cluster (tiny brute-force cases, edge cases)."""
    lat, powr, freq, models = make_tables(seed, M, F, S, B)
    states = make_states(seed, K, M, F, S, B, models, lo, min(hi, M, S), profile, local_sweep)
    reqs = make_requests(seed, R, M)
    return Cluster(name=f"custom{seed}", M=M, F=F, S=S, B=B, K=K, lat=lat, pow=powr,
                   freq_mhz=freq, models=models, states=states, requests=reqs, seed=seed)
