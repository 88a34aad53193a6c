"""The range claim behind the library's division-free round counts (fs_magic / fs_ceil_div_magic in
paper_2606_30391_b200/csrc/fs_common.cuh): for 1 <= n <= 256 and q <= 2^24,
    ceil(q / n) == umulhi(q - 1, ceil(2^32 / n)) + 1.
The arithmetic is restated here in 64-bit integers (no code is shared with the CUDA side) and checked where it
can break: the quotient is first wrong at the largest x = q - 1 with x mod n == n - 1, so every n is checked on
all such x in the top 2^20 of the range, on the last 2n values below 2^24, and on random q.  The admitted request
fields reach past 2^24 (O = (21*o_pred + 19) / 20 with o_pred < 2^24), where the identity does fail: the test
shows the first failures, which is why the placement kernel divides for real there (fs_place.cu)."""
from __future__ import annotations

import numpy as np

TOP = 1 << 24


def _magic(n: int) -> int:
    return 0 if n <= 1 else ((1 << 32) + n - 1) // n


def _ceil_div_magic(q: np.ndarray, n: int) -> np.ndarray:
    m = _magic(n)
    q = q.astype(np.uint64)
    if m == 0:
        return q
    x = np.where(q == 0, 0, q - 1).astype(np.uint64)
    return np.where(q == 0, 0, ((x * np.uint64(m)) >> np.uint64(32)) + np.uint64(1))


def test_exact_up_to_2_pow_24_for_every_divisor():
    rng = np.random.default_rng(7)
    for n in range(1, 257):
        lo = TOP - (1 << 20)
        first = lo + ((n - 1 - lo) % n)                       # x = q-1 with x mod n == n-1: worst residues
        x = np.arange(first, TOP, n, dtype=np.int64)
        q = np.concatenate([x + 1, np.arange(TOP - 2 * n, TOP + 1), rng.integers(0, TOP + 1, 20000), [0, 1, n, n + 1]])
        q = q[(q >= 0) & (q <= TOP)]
        want = (q + n - 1) // n
        assert np.array_equal(_ceil_div_magic(q, n).astype(np.int64), want), n


def test_first_failures_lie_beyond_2_pow_24():
    o_max = (21 * (TOP - 1) + 19) // 20                       # largest padded output length the ABI admits
    assert o_max == 17616076
    q = np.arange(TOP, o_max + 1, dtype=np.int64)
    firsts = {}
    for n in (252, 255, 256, 3):
        bad = q[_ceil_div_magic(q, n).astype(np.int64) != (q + n - 1) // n]
        firsts[n] = int(bad[0]) if len(bad) else None
    assert firsts[255] == 16909560 and firsts[252] == 17318448        # one round too many from there on
    assert firsts[256] is None and firsts[3] is None                   # powers of two never fail; small n fail far later
    assert int(_ceil_div_magic(np.array([16909560]), 255)[0]) == 66313 and -(-16909560 // 255) == 66312
