"""Pins of the oracle's transmission plan (Kuhn-Munkres assignment over e_uv = Bytes/BW) and of the
selective-migration rules (Appendix E).  CPU only."""
from __future__ import annotations

import itertools

import numpy as np
import pytest

import oracle
from paper_2606_30391_b200 import synth

f32 = np.float32


def _costs(bytes_mb, bw):
    t = (bytes_mb.astype(f32)[:, None] / bw.astype(f32)).astype(f32)
    return np.rint((t * f32(1000.0)).astype(f32)).astype(np.int64)


@pytest.mark.parametrize("seed", range(20))
def test_assignment_against_brute_force(seed):
    st = synth.Stream(seed, "assign")
    n = int(st.randint(1, 1, 7)[0])
    bytes_mb = st.urange(n, 1.0, 100.0).astype(f32)
    bw = st.urange(n * n, 1.0, 10.0).reshape(n, n).astype(f32)
    if seed % 3 == 0:
        bw = np.round(bw)                                     # many equal costs
        bytes_mb = np.round(bytes_mb / 10) * 10 + 10
    dst, tot = oracle.assign(bytes_mb, bw)
    c = _costs(bytes_mb, bw)
    best = min(sum(c[u, p[u]] for u in range(n)) for p in itertools.permutations(range(n)))
    assert sorted(dst) == list(range(n)) and tot == best == sum(c[u, dst[u]] for u in range(n))


@pytest.mark.parametrize("n", [1, 2, 8, 33, 120])
def test_assignment_against_scipy(n):
    from scipy.optimize import linear_sum_assignment
    bytes_mb, bw, _ = synth.make_migration(n, n, 0)
    dst, tot = oracle.assign(bytes_mb, bw)
    c = _costs(bytes_mb, bw)
    rows, cols = linear_sum_assignment(c)
    assert sorted(dst) == list(range(n)) and tot == int(c[rows, cols].sum()) == int(sum(c[u, dst[u]] for u in range(n)))


def test_assignment_by_hand():
    # two sources, two destinations: 1000 MB and 10 MB; staying costs nothing, the cross links are 10 MB/ms
    bw = np.array([[1e6, 10.0], [10.0, 1e6]], dtype=f32)
    dst, tot = oracle.assign(np.array([1000.0, 10.0], f32), bw)
    assert list(dst) == [0, 1] and tot == 1 + 0            # 1000 MB / 1e6 MB/ms = 1 us, 10 MB -> 0.01 us -> 0
    # if source 0 must leave (its own slot is slow), the big state takes the fast link
    bw = np.array([[1.0, 100.0], [10.0, 10.0]], dtype=f32)
    dst, tot = oracle.assign(np.array([1000.0, 10.0], f32), bw)
    assert list(dst) == [1, 0] and tot == 10000 + 1000     # 10 ms + 1 ms


def test_selective_migration_rules():
    """finish in place when close to completion; KV only when the link beats recomputation."""
    q = np.zeros(4, dtype=synth.MIG_REQ_DT)
    #      remaining  tokens  kv     bw    recompute
    q[0] = (5.0,      0.01,   900.0, 450.0, 50.0, (0, 0, 0))    # kv_tx 2 ms < 50: KV; mig ~2 ms < 5 remaining: migrate
    q[1] = (1.0,      0.01,   900.0, 450.0, 50.0, (0, 0, 0))    # almost done: finish locally
    q[2] = (500.0,    0.01,   900.0, 9.0,   50.0, (0, 0, 0))    # kv_tx 100 ms > 50: tokens only, recompute; migrate
    q[3] = (40.0,     0.01,   900.0, 9.0,   50.0, (0, 0, 0))    # 50 ms to rebuild > 40 ms left: finish locally
    flags, ms = oracle.migration_select(q)
    assert list(flags) == [3, 2, 1, 0]
    assert ms[0] == f32(f32(0.01) / f32(450.0)) + f32(2.0) and ms[2] == f32(f32(f32(0.01) / f32(9.0)) + f32(50.0))
