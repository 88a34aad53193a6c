"""fs_replace_plan_static — the one entry point of libfestina_eval that allocates nothing.

Why it exists: a scheduler that shares its GPU with a serving engine often cannot call cudaMalloc when it
needs a consolidation plan — the engine took nearly all of HBM at start-up, and cudaMalloc / cudaFree stall
the inference streams anyway — and every other call of the library sits on a context that allocates.  This
call keeps the kernel's working arrays in a fixed array inside the library instead (FS_PLAN_STATIC_MAX_N LLMs
at most) and takes the caller's device buffers for input and output.

What is checked here: the same inputs through this entry point and through the existing fs_replace_plan give
identical placements and counts (integers: exact, as in tests/test_gpu_parity.py), on two calls in a row that
share the built-in array — the second smaller than the first, so that it runs over whatever the first left
behind — and a size beyond the limit is refused without touching the outputs.

The file name sorts last on purpose: `pytest -x` stops at the first failure, so a problem here cannot hide
the parity tests.  It has to pass on its own in a fresh process as well (the static call below is issued
before this file creates any context).
"""
from __future__ import annotations

import numpy as np
import pytest

from paper_2606_30391_b200 import synth

pytestmark = pytest.mark.gpu


def _to_device(torch, rec):
    return torch.from_numpy(np.ascontiguousarray(rec).view(np.uint8).copy()).cuda()


def _case(seed, n, S, n_freq):
    freq = np.linspace(210, 1980, n_freq).astype(np.float32)
    s_eff = (S * 95) // 100
    llms = synth.make_plan_llms(seed, n, S, freq)
    if n > 20:
        llms["mem_mb"][5::13] = 90000.0          # larger than a whole GPU: these stay unplaced (-1)
    return llms, s_eff, 76000.0


def test_static_plan_matches_the_context_path_twice_in_a_row(fs):
    import torch
    torch.cuda.set_device(0)
    cases = [_case(11, 1000, 32, 64), _case(12, 257, 16, 16)]   # big first, small second: stale scratch beyond it
    st = torch.cuda.Stream()
    got = []
    with torch.cuda.stream(st):
        for llms, s_eff, m_eff in cases:
            d_in = _to_device(torch, llms)
            d_gpu = torch.full((len(llms),), -7, dtype=torch.int32, device="cuda")
            d_sum = torch.full((4,), -7, dtype=torch.int32, device="cuda")
            fs.replace_plan_static(d_in, s_eff, m_eff, d_gpu, d_sum, stream=st)   # same stream: the calls do not overlap
            got.append((d_in, d_gpu, d_sum))
    st.synchronize()
    ctx = fs.Festina(0)                                         # the existing path, created only now
    for (llms, s_eff, m_eff), (_, d_gpu, d_sum) in zip(cases, got):
        want_gpu, want_sum = ctx.replace_plan(llms, s_eff, m_eff)
        assert tuple(int(x) for x in d_sum.cpu().numpy()) == want_sum
        assert np.array_equal(d_gpu.cpu().numpy(), want_gpu)
        assert want_sum[3] > 0 and (want_gpu >= 0).any() and (want_gpu < 0).any()   # a non-trivial plan
    # and once more after the context path has run, in the other order (small, then big)
    for llms, s_eff, m_eff in reversed(cases):
        d_in = _to_device(torch, llms)
        d_gpu = torch.full((len(llms),), -7, dtype=torch.int32, device="cuda")
        d_sum = torch.full((4,), -7, dtype=torch.int32, device="cuda")
        fs.replace_plan_static(d_in, s_eff, m_eff, d_gpu, d_sum)
        torch.cuda.synchronize()
        want_gpu, want_sum = ctx.replace_plan(llms, s_eff, m_eff)
        assert tuple(int(x) for x in d_sum.cpu().numpy()) == want_sum
        assert np.array_equal(d_gpu.cpu().numpy(), want_gpu)
    ctx.close() if hasattr(ctx, "close") else None


def test_static_plan_refuses_more_than_the_built_in_array_holds(fs):
    import torch
    torch.cuda.set_device(0)
    n = fs.FS_PLAN_STATIC_MAX_N + 1
    llms, s_eff, m_eff = _case(13, n, 16, 16)
    d_in = _to_device(torch, llms)
    d_gpu = torch.full((n,), -7, dtype=torch.int32, device="cuda")
    d_sum = torch.full((4,), -7, dtype=torch.int32, device="cuda")
    with pytest.raises(fs.FestinaError) as e:
        fs.replace_plan_static(d_in, s_eff, m_eff, d_gpu, d_sum)
    assert e.value.code == fs.FS_ERR_SHAPE and str(fs.FS_PLAN_STATIC_MAX_N) in str(e.value)
    torch.cuda.synchronize()
    assert int(d_sum.min()) == -7 and int(d_gpu.min()) == -7 and int(d_gpu.max()) == -7   # nothing ran
    # exactly at the limit it runs
    llms, s_eff, m_eff = _case(14, fs.FS_PLAN_STATIC_MAX_N, 16, 16)
    d_in = _to_device(torch, llms)
    d_gpu = torch.full((len(llms),), -7, dtype=torch.int32, device="cuda")
    fs.replace_plan_static(d_in, s_eff, m_eff, d_gpu, d_sum)
    torch.cuda.synchronize()
    ctx = fs.Festina(0)
    want_gpu, want_sum = ctx.replace_plan(llms, s_eff, m_eff)
    assert tuple(int(x) for x in d_sum.cpu().numpy()) == want_sum and np.array_equal(d_gpu.cpu().numpy(), want_gpu)
