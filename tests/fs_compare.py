"""Element-by-element comparison of CUDA results with oracle results (tests only).

Bar (BASELINE.json north_star): chosen GPU / SM share / frequency / batch indices bit-exact,
energies and latencies within 1e-5 relative error.  DESIGN.md "Numerics" promises more (both
sides round every operation identically), so `exact=True` also demands bitwise-equal floats.
"""
from __future__ import annotations

import numpy as np

RTOL = 1e-5


def _float_close(a, b, name, exact):
    a = np.asarray(a, dtype=np.float32)
    b = np.asarray(b, dtype=np.float32)
    same_inf = np.isinf(a) & np.isinf(b) & (np.sign(a) == np.sign(b))
    if exact:
        bad = ~((a.view(np.uint32) == b.view(np.uint32)) | ((a == 0) & (b == 0)))
    else:
        with np.errstate(invalid="ignore"):
            bad = ~(same_inf | (np.abs(a - b) <= RTOL * np.maximum(np.abs(a), np.abs(b))))
    if bad.any():
        i = int(np.flatnonzero(bad.reshape(len(a), -1).any(axis=1))[0])
        raise AssertionError(f"{name}: {int(bad.sum())} mismatches, first at record {i}: cuda={a[i]!r} oracle={b[i]!r}")


def _int_equal(a, b, name):
    a = np.asarray(a)
    b = np.asarray(b)
    bad = a != b
    if bad.any():
        i = int(np.flatnonzero(bad.reshape(len(a), -1).any(axis=1))[0])
        raise AssertionError(f"{name}: {int(bad.sum())} mismatches, first at record {i}: cuda={a[i]!r} oracle={b[i]!r}")


def assert_placement_equal(got, ref, exact=True):
    assert len(got) == len(ref)
    for f in ("gpu", "sigma", "phi", "beta", "f_req", "flat"):
        _int_equal(got[f], ref[f], f"placement.{f}")
    for f in ("energy_mj", "ttft_ms", "tbt_ms"):
        _float_close(got[f], ref[f], f"placement.{f}", exact)


def assert_local_equal(got, ref, exact=True):
    assert len(got) == len(ref)
    for f in ("phi", "f_req", "sigma", "beta", "flat"):
        _int_equal(got[f], ref[f], f"local.{f}")
    for f in ("cost", "energy_mj", "power_w"):
        _float_close(got[f], ref[f], f"local.{f}", exact)


def assert_consol_equal(got, ref, exact=True):
    assert len(got) == len(ref)
    for f in ("dst", "phi"):
        _int_equal(got[f], ref[f], f"consol.{f}")
    for f in ("score_mj", "saving_mj"):
        _float_close(got[f], ref[f], f"consol.{f}", exact)


def assert_tasks_equal(got, ref):
    assert len(got) == len(ref)
    for f in ("rank", "admitted"):
        _int_equal(got[f], ref[f], f"tasks.{f}")
    for f in ("score", "latency_ms"):
        _float_close(got[f], ref[f], f"tasks.{f}", True)
