"""CPU oracle of the Festina decision arithmetic — TEST INFRASTRUCTURE, not the product.

ctypes wrapper around oracle/festina_oracle.cpp (plain C++17, written from PAPER.md; see that
file's header for the pins).  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
`--impl reference` legs may import this package; the CUDA path never does.  Inputs are numpy
record arrays in the layout of include/festina_eval.h (the seeded generator
paper_2606_30391_b200/synth.py produces them); outputs are numpy record arrays.
"""
from __future__ import annotations

import ctypes as C

import numpy as np

from .build import build as _build

_PLACEMENT_DT = np.dtype(
    [("gpu", "<i4"), ("sigma", "<i2"), ("phi", "<i2"), ("beta", "<i2"), ("f_req", "<i2"),
     ("energy_mj", "<f4"), ("ttft_ms", "<f4"), ("tbt_ms", "<f4"), ("flat", "<u4"), ("_pad", "<u4")])
_LOCAL_DT = np.dtype(
    [("phi", "<i2"), ("f_req", "<i2"), ("sigma", "u1", (4,)), ("beta", "u1", (4, 2)),
     ("cost", "<f4"), ("energy_mj", "<f4"), ("power_w", "<f4"), ("flat", "<u4"),
     ("_pad", "<u4", (4,))])
_CONSOL_DT = np.dtype([("dst", "<i4"), ("phi", "<i4"), ("score_mj", "<f4"), ("saving_mj", "<f4")])

_LLM_PROFILE_DT = np.dtype([("sigma_p", "<i2"), ("phi_p", "<i2"), ("sigma_d", "<i2"), ("phi_d", "<i2"),
                            ("t_p_ms", "<f4"), ("t_d_ms", "<f4"), ("p_p_w", "<f4"), ("p_d_w", "<f4"),
                            ("sm_units", "<f4"), ("need_units", "<i2"), ("phi_l", "<i2"), ("t_l_ms", "<f4"),
                            ("e_l_mj", "<f4"), ("mem_mb", "<f4"), ("_pad", "<u4")])
_TASK_OUT_DT = np.dtype([("score", "<f4"), ("latency_ms", "<f4"), ("rank", "<i4"), ("admitted", "<i4")])

OBJ_ENERGY, OBJ_POWER, SPLIT_EXHAUSTIVE, SPLIT_MINSM = 0, 1, 0, 2

_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build())
        _lib.fo_slot.restype = C.c_int
        _lib.fo_slot.argtypes = [C.c_int] * 4 + [C.c_void_p] * 2 + [C.c_int] * 5 + [C.c_uint32, C.c_float, C.c_float, C.c_void_p, C.c_void_p]
    return _lib


def _p(a: np.ndarray):
    assert a.flags["C_CONTIGUOUS"]
    return C.c_void_p(a.ctypes.data)


def _tables(lat: np.ndarray, pow_: np.ndarray):
    assert lat.dtype == np.float32 and pow_.dtype == np.float32 and lat.shape == pow_.shape
    M, P, F, S, B = lat.shape
    assert P == 2
    return (C.c_int(M), C.c_int(F), C.c_int(S), C.c_int(B), _p(lat), _p(pow_))


def place_batch(lat, pow_, models, states, reqs, nthreads: int = 1) -> np.ndarray:
    """fs_place_batch by definition (PAPER.md; readings s2-s6)."""
    out = np.zeros(len(reqs), dtype=_PLACEMENT_DT)
    lib().fo_place_batch(*_tables(lat, pow_), _p(models), C.c_int(len(states)), _p(states),
                         C.c_int(len(reqs)), _p(reqs), _p(out), C.c_int(nthreads))
    return out


def dispatch(lat, pow_, models, states, reqs, nthreads: int = 1) -> np.ndarray:
    """The paper's three-phase dispatcher at (F_curr, SM_free) (Eq. 2-3)."""
    out = np.zeros(len(reqs), dtype=_PLACEMENT_DT)
    lib().fo_dispatch(*_tables(lat, pow_), _p(models), C.c_int(len(states)), _p(states),
                      C.c_int(len(reqs)), _p(reqs), _p(out), C.c_int(nthreads))
    return out


def dispatch_commit(lat, pow_, models, states, reqs):
    """The dispatcher with the sequential commit pass (reading s34 of PAPER.md lines 214-218):
    returns (placements, the state records after the last commit)."""
    out = np.zeros(len(reqs), dtype=_PLACEMENT_DT)
    st = np.array(states, copy=True)
    lib().fo_dispatch_commit(*_tables(lat, pow_), _p(models), C.c_int(len(st)), _p(st),
                             C.c_int(len(reqs)), _p(reqs), _p(out))
    return out, st


def local_config(lat, pow_, states, flags: int, gpu_ids=None, nthreads: int = 1) -> np.ndarray:
    """fs_local_config by definition (Fig. 8 step 3)."""
    if gpu_ids is None:
        n, ids = len(states), C.c_void_p(0)
    else:
        gpu_ids = np.ascontiguousarray(gpu_ids, dtype=np.int32)
        n, ids = len(gpu_ids), _p(gpu_ids)
    out = np.zeros(n, dtype=_LOCAL_DT)
    lib().fo_local_config(*_tables(lat, pow_), _p(states), C.c_int(n), ids, C.c_uint32(flags),
                          _p(out), C.c_int(nthreads))
    return out


def consolidate(lat, pow_, models, states, p_idle_w, horizon_ms, mem_cap_mb, delta_pct,
                nthreads: int = 1) -> np.ndarray:
    """fs_consolidate by definition (PAPER.md, 623; readings s17-s20)."""
    out = np.zeros(len(states), dtype=_CONSOL_DT)
    lib().fo_consolidate(*_tables(lat, pow_), _p(models), C.c_int(len(states)), _p(states),
                         C.c_float(p_idle_w), C.c_float(horizon_ms), C.c_float(mem_cap_mb),
                         C.c_int(delta_pct), _p(out), C.c_int(nthreads))
    return out


def batch_tasks(lat, pow_, states, off, tasks, gpu_ids=None, nthreads: int = 1) -> np.ndarray:
    """Local scheduler steps 1-2 by definition (Eq. 4, Fig. 8)."""
    off = np.ascontiguousarray(off, dtype=np.int32)
    n = len(off) - 1
    ids = C.c_void_p(0)
    if gpu_ids is not None:
        gpu_ids = np.ascontiguousarray(gpu_ids, dtype=np.int32)
        assert len(gpu_ids) == n
        ids = _p(gpu_ids)
    out = np.zeros(len(tasks), dtype=_TASK_OUT_DT)
    lib().fo_batch_tasks(*_tables(lat, pow_), _p(states), C.c_int(n), ids, _p(off),
                         _p(np.ascontiguousarray(tasks)), _p(out), C.c_int(nthreads))
    return out


def llm_profile(lat, pow_, models, llms, nthreads: int = 1) -> np.ndarray:
    """Algorithm 1 phase 1 by definition (PAPER.md, 337-339, Eq. 8, Little's law)."""
    out = np.zeros(len(llms), dtype=_LLM_PROFILE_DT)
    lib().fo_llm_profile(*_tables(lat, pow_), _p(models), C.c_int(len(llms)), _p(np.ascontiguousarray(llms)),
                         _p(out), C.c_int(nthreads))
    return out


def ewr(gpu_of, f_mhz, t_ms, K: int):
    """Energy Waste Ratio, Eq. 5-7: returns (F_g [K], E_waste, E_optimal, EWR)."""
    gpu_of = np.ascontiguousarray(gpu_of, dtype=np.int32)
    f_mhz = np.ascontiguousarray(f_mhz, dtype=np.float32)
    t_ms = np.ascontiguousarray(t_ms, dtype=np.float32)
    fg = np.zeros(max(K, 1), dtype=np.float32)
    out = np.zeros(3, dtype=np.float64)
    lib().fo_ewr(C.c_int(len(gpu_of)), _p(gpu_of), _p(f_mhz), _p(t_ms), C.c_int(K), _p(fg), _p(out))
    return fg[:K], float(out[0]), float(out[1]), float(out[2])


def replace_plan(llms, s_eff: int, m_eff: float):
    """Algorithm 1 phases 2-3: returns (gpu_of [n], (N_sm, N_mem, N_min, N_active))."""
    llms = np.ascontiguousarray(llms)
    gpu_of = np.full(len(llms), -1, dtype=np.int32)
    summ = np.zeros(4, dtype=np.int32)
    lib().fo_replace_plan(C.c_int(len(llms)), _p(llms), C.c_int(s_eff), C.c_float(m_eff), _p(gpu_of), _p(summ))
    return gpu_of, tuple(int(x) for x in summ)


def assign(bytes_mb, bw_mb_per_ms):
    """Minimum-cost source -> destination assignment, costs in whole microseconds."""
    bytes_mb = np.ascontiguousarray(bytes_mb, dtype=np.float32)
    bw = np.ascontiguousarray(bw_mb_per_ms, dtype=np.float32)
    n = len(bytes_mb)
    assert bw.shape == (n, n)
    dst = np.full(max(n, 1), -1, dtype=np.int32)
    tot = np.zeros(1, dtype=np.int64)
    lib().fo_assign(C.c_int(n), _p(bytes_mb), _p(bw), _p(dst), _p(tot))
    return dst[:n], int(tot[0])


def migration_select(reqs):
    """Finish locally vs migrate, tokens vs KV: returns (flags u8, migration ms)."""
    reqs = np.ascontiguousarray(reqs)
    out = np.zeros(max(len(reqs), 1), dtype=np.uint8)
    ms = np.zeros(max(len(reqs), 1), dtype=np.float32)
    lib().fo_migration_select(C.c_int(len(reqs)), _p(reqs), _p(out), _p(ms))
    return out[:len(reqs)], ms[:len(reqs)]


def slot(lat, pow_, m, p, phi, sigma, beta, q, wait, slo):
    """The shared slot rule: returns (ok, t, e)."""
    t = C.c_float(0)
    e = C.c_float(0)
    ok = lib().fo_slot(*_tables(lat, pow_), m, p, phi, sigma, beta, C.c_uint32(q),
                       C.c_float(wait), C.c_float(slo), C.byref(t), C.byref(e))
    return bool(ok), np.float32(t.value), np.float32(e.value)


def gpu_freq_floor(lat, pow_, state_rec: np.ndarray) -> int:
    s = np.ascontiguousarray(state_rec).reshape(1)
    return int(lib().fo_gpu_freq_floor(*_tables(lat, pow_), _p(s)))


def tenant_fmin(lat, pow_, state_rec: np.ndarray, i: int) -> int:
    s = np.ascontiguousarray(state_rec).reshape(1)
    return int(lib().fo_tenant_fmin(*_tables(lat, pow_), _p(s), C.c_int(i)))
