"""Parity of the CUDA path (through the C ABI) with the CPU oracle, element by element, on the
same seeded inputs.  Everything here needs a B200: `-m gpu`."""
from __future__ import annotations

import os

import numpy as np
import pytest

import fs_compare as cmp
import fs_util as U
import oracle
from paper_2606_30391_b200 import synth
import bench_work

pytestmark = pytest.mark.gpu

ALL_FLAGS = [0, 1, 2, 3]


@pytest.fixture(scope="module")
def ctx(fs):
    c = fs.Festina(0)
    yield c
    c.close()


NTHREADS = os.cpu_count() or 8


def _oracle_place(cl, reqs=None, nthreads=NTHREADS):
    return oracle.place_batch(cl.lat, cl.pow, cl.models, cl.states, cl.requests if reqs is None else reqs, nthreads)


def _oracle_local(cl, flags, ids=None, nthreads=NTHREADS):
    return oracle.local_config(cl.lat, cl.pow, cl.states, flags, ids, nthreads)


def _oracle_consol(cl, nthreads=NTHREADS):
    p = cl.params
    return oracle.consolidate(cl.lat, cl.pow, cl.models, cl.states, p.p_idle_w, p.horizon_ms,
                              p.mem_cap_mb, p.delta_pct, nthreads)


def _check_all(ctx, cl, local=True, consol=True):
    ctx.load_cluster(cl)
    if cl.R:
        got = ctx.place_batch(cl.requests)
        cmp.assert_placement_equal(got, _oracle_place(cl))
    if local:
        for fl in ALL_FLAGS:
            cmp.assert_local_equal(ctx.local_config(fl), _oracle_local(cl, fl))
    if consol:
        cmp.assert_consol_equal(ctx.consolidate(), _oracle_consol(cl))


# ---- config 0 and ragged small clusters: everything, element by element ----------------------
def test_tiny_config_all_entry_points(ctx):
    cl = synth.make_cluster("tiny")
    _check_all(ctx, cl)
    got = ctx.place_batch(cl.requests)
    assert (got["gpu"] >= 0).sum() > 200          # not a degenerate all-infeasible case


@pytest.mark.parametrize("seed", range(12))
def test_ragged_dims(ctx, seed):
    """Dims that are not multiples of the warp / tile sizes, several tenants, ragged tails."""
    st = synth.Stream(seed, "dims")
    K = int(st.randint(1, 1, 70)[0]); M = int(st.randint(1, 1, 9)[0])
    F = int(st.randint(1, 1, 70)[0]); S = int(st.randint(1, 1, 20)[0]); B = int(st.randint(1, 1, 40)[0])
    cl = synth.make_custom(seed=100 + seed, K=K, M=M, F=F, S=S, B=B, R=97, lo=1, hi=4)
    _check_all(ctx, cl)


@pytest.mark.parametrize("seed", range(6))
def test_tie_heavy_tables(ctx, seed):
    """Tables quantised to a few powers of two: exact ties everywhere, lowest flat index wins."""
    cl = U.tie_heavy(synth.make_custom(seed=200 + seed, K=9, M=3, F=12, S=6, B=5, R=64), seed)
    cl.requests["slo_ttft_ms"] = 1e9
    cl.requests["slo_tbt_ms"] = 1e9
    cl.states["t"]["slo_ms"][...] = 1e9
    _check_all(ctx, cl)


def test_duplicate_models_on_one_gpu(ctx):
    """The join target is the LOWEST slot holding the model."""
    cl = synth.make_custom(seed=31, K=6, M=2, F=8, S=8, B=8, R=32, lo=2, hi=2)
    cl.states["t"]["model"][:, 1] = cl.states["t"]["model"][:, 0]
    _check_all(ctx, cl)


def test_edge_cases(ctx):
    cl = synth.make_custom(seed=41, K=12, M=3, F=10, S=8, B=8, R=40, lo=1, hi=4)
    cl.states["n_res"][0] = 0                       # inactive GPU
    cl.states["t"]["q"][1] = 0                      # all queues empty
    cl.states["t"]["sigma"][2, :] = 1               # 4 tenants x 2 units = S: no free SMs
    cl.states["n_res"][2] = 4
    cl.states["t"]["model"][2] = [0, 1, 2, 0]
    cl.states["t"]["beta"][3, :, 1] = cl.B - 1      # decode bucket already at the last level
    cl.requests["L"][0] = 0
    cl.requests["o_pred"][1] = 0
    cl.requests["L"][2] = 1
    cl.requests["slo_ttft_ms"][3] = 0.0             # nothing feasible
    cl.requests["slo_tbt_ms"][4] = 0.0
    cl.requests["L"][5] = 4096
    cl.requests["o_pred"][5] = 4096
    _check_all(ctx, cl)
    got = ctx.place_batch(cl.requests)
    assert got["gpu"][3] == -1 and np.isinf(got["energy_mj"][3]) and got["flat"][3] == 0xFFFFFFFF


@pytest.mark.parametrize("seed", range(4))
def test_ttft_deadline_on_the_rounding_boundary(ctx, seed):
    """slo_ttft set to fl(wait + t0) of a real candidate, and to its float neighbours, so that the
    deadline test sits exactly on a rounding boundary (the dense kernel's threshold T*)."""
    cl = synth.make_custom(seed=300 + seed, K=40, M=6, F=48, S=12, B=16, R=192, lo=1, hi=3)
    st = synth.Stream(seed, "boundary")
    f32 = np.float32
    for r in range(cl.R):
        rq = cl.requests[r]
        m, L = int(rq["model"]), int(rq["L"])
        k = int(st.randint(1, 0, cl.K - 1)[0]); sg = int(st.randint(1, 0, cl.S - 1)[0])
        phi = int(st.randint(1, 0, cl.F - 1)[0])
        g = cl.states[k]
        cold = m not in [int(g["t"][i]["model"]) for i in range(int(g["n_res"]))]
        wait = f32(g["t_avail_ms"]) + (f32(cl.models["load_ms"][m]) if cold else f32(0))
        b0 = min(L, cl.B) - 1
        t0 = f32(-(-L // (b0 + 1))) * cl.lat[m, 0, phi, sg, b0]
        edge = f32(f32(wait) + f32(t0))
        which = r % 3
        cl.requests["slo_ttft_ms"][r] = [edge, np.nextafter(edge, f32(-np.inf)), np.nextafter(edge, f32(np.inf))][which]
        if r % 7 == 0:                                  # tiny waits: t0 dominates the sum
            cl.states["t_avail_ms"][k] = f32(1e-6) * f32(r + 1)
    cl.models["load_ms"][::2] = 0.0                     # wait can be exactly t_avail
    _check_all(ctx, cl, local=False, consol=False)


@pytest.mark.parametrize("B", [4, 12, 64, 256])
def test_local_queue_depths_up_to_2_pow_24(ctx, B):
    """rounds = ceil(q/(beta+1)) for q from 1 to 2^24-1 (the kernel divides by multiply-high)."""
    cl = synth.make_custom(seed=500 + B, K=48, M=5, F=6, S=4, B=B, R=0, lo=1, hi=4)
    st = synth.Stream(B, "bigq")
    q = st.randint(cl.K * 8, 0, 24).reshape(cl.K, 4, 2)
    q = (2 ** q.astype(np.int64)) - st.randint(cl.K * 8, 0, 3).reshape(cl.K, 4, 2)
    cl.states["t"]["q"][...] = np.clip(q, 0, 2 ** 24 - 1).astype(np.uint32)
    cl.states["t"]["slo_ms"][...] = 1e30
    _check_all(ctx, cl, consol=False)


def test_padded_output_lengths_past_2_pow_24(ctx):
    """o_pred up to 2^24-1 pads to O = (21*o_pred+19)/20 > 2^24, beyond the range in which the placement kernel's
    multiply-high round count is exact (tests/test_magic_division.py): decode buckets 252 / 255 of a B = 256
    table joined by requests whose O sits on and around the first values at which the shortcut is one round off
    (16,909,560 for 255; 17,318,448 for 252), plus prompts L near 2^24 for the prefill shortcut."""
    cl = synth.make_custom(seed=77, K=24, M=2, F=6, S=4, B=256, R=160, lo=1, hi=2)
    st = synth.Stream(77, "bigO")
    cl.states["t"]["beta"][:, :, 1] = np.array([250, 253, 251, 254, 255, 0], dtype=np.uint8)[st.randint(cl.K * 4, 0, 5)].reshape(cl.K, 4)
    cl.states["t"]["q"][:, :, 1] = 1 + st.randint(cl.K * 4, 0, 1000).reshape(cl.K, 4).astype(np.uint32)
    cl.states["t"]["sigma"][...] = 0                     # free shares everywhere
    cl.states["t"]["slo_ms"][...] = 1e30
    cl.states["mem_free_mb"] = 1e30
    cl.models["kv_mb_per_token"] = 1e-9
    cl.requests["slo_ttft_ms"] = 1e30
    cl.requests["slo_tbt_ms"] = 1e30
    crit = []
    for O in (16909560, 17318448, 1 << 24, (1 << 24) + 1, 17616076):
        crit += [(20 * (O + d)) // 21 + e for d in (-1, 0, 1, 255) for e in (0, 1)]     # o_pred with pad near O
    o = np.array(crit + list(2 ** 24 - 1 - st.randint(cl.R, 0, 900000)), dtype=np.int64)[:cl.R]
    cl.requests["o_pred"] = np.clip(o, 0, 2 ** 24 - 1).astype(np.uint32)
    cl.requests["L"][::3] = (2 ** 24 - 1 - st.randint(len(cl.requests["L"][::3]), 0, 70000)).astype(np.uint32)
    pad = (21 * cl.requests["o_pred"].astype(np.int64) + 19) // 20
    assert (pad == 16909560).any() and (pad == 17318448).any() and (pad > 2 ** 24).sum() > 100
    ctx.load_cluster(cl)
    got = ctx.place_batch(cl.requests)
    ref = _oracle_place(cl)
    cmp.assert_placement_equal(got, ref)
    warm = cl.states["t"]["model"][got["gpu"], 0] == cl.requests["model"]
    assert (got["gpu"] >= 0).all() and (got["beta"] >= 251).sum() > 20 and warm.sum() > 20     # joined the deep buckets
    cmp.assert_placement_equal(ctx.dispatch(cl.requests), _oracle_dispatch(cl))


def test_empty_inputs(ctx):
    cl = synth.make_custom(seed=5, K=4, M=2, F=4, S=4, B=4, R=8)
    ctx.load_cluster(cl)
    assert len(ctx.place_batch(cl.requests[:0])) == 0
    assert len(ctx.local_config(0, gpu_ids=np.zeros(0, np.int32))) == 0
    ctx.set_gpu_state(cl.states[:0])                # K = 0
    got = ctx.place_batch(cl.requests)
    assert (got["gpu"] == -1).all() and np.isinf(got["energy_mj"]).all()
    assert len(ctx.consolidate()) == 0


def test_local_gpu_id_subset(ctx):
    cl = synth.make_custom(seed=6, K=20, M=4, F=16, S=8, B=16, R=0, lo=1, hi=4)
    ctx.load_cluster(cl)
    ids = np.array([19, 0, 7, 7, 3], dtype=np.int32)
    for fl in ALL_FLAGS:
        cmp.assert_local_equal(ctx.local_config(fl, gpu_ids=ids), _oracle_local(cl, fl, ids))


def test_device_buffers_and_stream(ctx):
    """FS_DEVICE pointers on a non-default torch stream give the same bytes as FS_HOST."""
    import torch
    cl = synth.make_cluster("tiny")
    dev = torch.device("cuda:0")
    tb = lambda a: torch.from_numpy(np.ascontiguousarray(a).view(np.uint8).reshape(-1)).to(dev)
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        lat, pw = torch.from_numpy(cl.lat).to(dev), torch.from_numpy(cl.pow).to(dev)
        ctx.load_profiles(lat, pw, tb(cl.freq_mhz), tb(cl.models), cl.params, stream=s)
        ctx.set_gpu_state(tb(cl.states), stream=s)
        out = torch.empty(cl.R * 32, dtype=torch.uint8, device=dev)
        ctx.place_batch(tb(cl.requests), out=out, stream=s)
        lout = torch.empty(cl.K * 48, dtype=torch.uint8, device=dev)
        ctx.local_config(0, n=cl.K, out=lout, stream=s)
        cout = torch.empty(cl.K * 16, dtype=torch.uint8, device=dev)
        ctx.consolidate(out=cout, stream=s)
    s.synchronize()
    cmp.assert_placement_equal(out.cpu().numpy().view(synth.PLACEMENT_DT), _oracle_place(cl))
    cmp.assert_local_equal(lout.cpu().numpy().view(synth.LOCAL_CFG_DT), _oracle_local(cl, 0))
    cmp.assert_consol_equal(cout.cpu().numpy().view(synth.CONSOL_DT), _oracle_consol(cl))


# ---- error behaviour -------------------------------------------------------------------------
def test_errors(fs):
    c = fs.Festina(0)
    cl = synth.make_custom(seed=8, K=4, M=2, F=4, S=4, B=4, R=8)
    with pytest.raises(fs.FestinaError) as e:
        c.set_gpu_state(cl.states)                  # before fs_load_profiles
    assert e.value.code == fs.FS_ERR_STATE
    c.load_profiles(cl.lat, cl.pow, cl.freq_mhz, cl.models, cl.params)
    with pytest.raises(fs.FestinaError) as e:
        c.place_batch(cl.requests)                  # before fs_set_gpu_state
    assert e.value.code == fs.FS_ERR_STATE
    bad = cl.states.copy()
    bad["t"]["model"][1, 0] = 99                    # model index out of range
    c.set_gpu_state(bad)
    with pytest.raises(fs.FestinaError) as e:       # sticky flag surfaces on the next call
        c.place_batch(cl.requests)
    assert e.value.code == fs.FS_ERR_RANGE
    # the invalid GPU is treated as inactive; results equal the oracle's on the cleaned state
    clean = cl.states.copy()
    clean["n_res"][1] = 0
    got = c.place_batch(cl.requests)
    ref = oracle.place_batch(cl.lat, cl.pow, cl.models, clean, cl.requests)
    cmp.assert_placement_equal(got, ref)
    breq = cl.requests.copy()
    breq["model"][2] = -3
    with pytest.raises(fs.FestinaError) as e:
        c.place_batch(breq)
    assert e.value.code == fs.FS_ERR_RANGE
    with pytest.raises(fs.FestinaError) as e:
        big = synth.make_custom(seed=8, K=1, M=1, F=2, S=40, B=2, R=0)   # S > FS_MAX_S
        c.load_profiles(big.lat, big.pow, big.freq_mhz, big.models, big.params)
    assert e.value.code == fs.FS_ERR_SHAPE
    c.close()


# ---- BASELINE.json configs at full size ----------------------------------------------------
def test_rack_full(ctx):
    cl = synth.make_cluster("rack")
    ctx.load_cluster(cl)
    got = ctx.place_batch(cl.requests)
    cmp.assert_placement_equal(got, _oracle_place(cl))
    # the Poisson dispatch ticks (variable R per call) give the same decisions as one call
    ticks = synth.arrival_ticks(cl.seed, cl.R, 64)
    parts, o = [], 0
    for n in ticks:
        parts.append(ctx.place_batch(cl.requests[o:o + n]))
        o += n
    cmp.assert_placement_equal(np.concatenate(parts), got)
    for fl in ALL_FLAGS:
        cmp.assert_local_equal(ctx.local_config(fl), _oracle_local(cl, fl))
    cmp.assert_consol_equal(ctx.consolidate(), _oracle_consol(cl))


def test_pod_full_size(ctx):
    """configs[2] in the launch configuration bench.py times: ALL 65,536 placements and every GPU's local
    configuration under all four flag combinations, element by element against the oracle (the oracle scores
    the dense grid of 6.9e10 candidates: about a minute on the box's host cores)."""
    cl = synth.make_cluster("pod")
    ctx.load_cluster(cl)
    got = ctx.place_batch(cl.requests)
    cmp.assert_placement_equal(got, _oracle_place(cl))
    assert (got["gpu"] >= 0).mean() > 0.9
    for fl in ALL_FLAGS:
        cmp.assert_local_equal(ctx.local_config(fl), _oracle_local(cl, fl))


def test_local_sweep_full_size(ctx):
    """configs[3]: all 4,096 GPUs under all four flag combinations."""
    cl = synth.make_cluster("local")
    ctx.load_cluster(cl)
    for fl in ALL_FLAGS:
        got = ctx.local_config(fl)
        assert len(got) == cl.K
        cmp.assert_local_equal(got, _oracle_local(cl, fl))
        assert (got["phi"] >= 0).mean() > 0.5


def test_consolidation_full_size(ctx):
    cl = synth.make_cluster("consol")
    ctx.load_cluster(cl)
    got = ctx.consolidate()
    cmp.assert_consol_equal(got, _oracle_consol(cl))
    assert (got["dst"] >= 0).mean() > 0.5


# ---- local scheduler steps 1-2: priority score + batching (fs_batch_tasks) --------------------
def _oracle_tasks(cl, off, tasks, ids=None):
    return oracle.batch_tasks(cl.lat, cl.pow, cl.states, off, tasks, ids, 8)


@pytest.mark.parametrize("seed", range(8))
def test_batch_tasks_small_clusters(ctx, seed):
    """0..130 tasks per GPU (empty lists, one task, non-powers of two, > 4 warps of tasks)."""
    cl = synth.make_custom(seed=800 + seed, K=23, M=4, F=9, S=[4, 7, 10, 16][seed % 4], B=12, R=0)
    off, tasks = synth.make_tasks(seed, cl.K, cl.M, cl.S, cl.B, 0, 130)
    if seed % 2:                                    # heavy exact ties in the score
        tasks["slack_ms"] = 64.0; tasks["age_ms"] = 0.0; tasks["beta"] = tasks["beta"] % 2
        tasks["model"] = 0; tasks["sigma"] = tasks["sigma"] % 2
    ctx.load_cluster(cl)
    cmp.assert_tasks_equal(ctx.batch_tasks(off, tasks), _oracle_tasks(cl, off, tasks))


def test_batch_tasks_limits_and_subset(ctx):
    cl = synth.make_custom(seed=811, K=6, M=3, F=6, S=16, B=8, R=0)
    off, tasks = synth.make_tasks(11, 3, cl.M, cl.S, cl.B, 1024, 1024)      # FS_MAX_TASKS per GPU
    tasks["mem_mb"] *= 0.01                          # let many tasks fit the memory budget
    ids = np.array([5, 0, 5], dtype=np.int32)
    ctx.load_cluster(cl)
    got = ctx.batch_tasks(off, tasks, gpu_ids=ids)
    cmp.assert_tasks_equal(got, _oracle_tasks(cl, off, tasks, ids))
    assert got["admitted"].sum() > 3
    assert len(ctx.batch_tasks(np.zeros(1, np.int32), tasks[:0])) == 0      # no GPUs, no tasks


def test_batch_tasks_fig8(ctx):
    """The worked table of Fig. 8 steps 1-2 through the CUDA path."""
    from test_oracle_batching import _fig8_cluster
    lat, pw, st, tasks, names, fig = _fig8_cluster(mem_free=1e6)
    M, _, F, S, B = lat.shape
    models = np.zeros(M, dtype=synth.MODEL_INFO_DT)
    ctx.load_profiles(lat, pw, np.ones(F, np.float32), models, synth.Params())
    ctx.set_gpu_state(st)
    out = ctx.batch_tasks([0, 6], tasks)
    assert [names[i] for i in np.argsort(out["rank"])] == ["D1", "D3", "D2", "P1", "P3", "P2"]
    assert {nm: int(out["admitted"][i]) for i, nm in enumerate(names)} == \
        {"D1": 1, "D3": 1, "D2": 1, "P1": 0, "P3": 1, "P2": 0}


def test_batch_tasks_errors(fs):
    c = fs.Festina(0)
    cl = synth.make_custom(seed=812, K=4, M=2, F=4, S=4, B=4, R=0)
    off, tasks = synth.make_tasks(12, cl.K, cl.M, cl.S, cl.B, 3, 9)
    c.load_cluster(cl)
    bad = tasks.copy()
    bad["sigma"][off[2]] = 9                         # share index out of range on GPU 2
    with pytest.raises(fs.FestinaError) as e:
        c.batch_tasks(off, bad)
    assert e.value.code == fs.FS_ERR_RANGE
    with pytest.raises(fs.FestinaError) as e:
        c.batch_tasks(off, tasks, gpu_ids=np.array([0, 1, 99, 3], np.int32))
    assert e.value.code == fs.FS_ERR_RANGE
    got = c.batch_tasks(off, tasks)                  # clean call afterwards
    cmp.assert_tasks_equal(got, oracle.batch_tasks(cl.lat, cl.pow, cl.states, off, tasks))
    c.close()


def test_batch_tasks_pod_size(ctx):
    """1,024 GPUs x 10-100 queued tasks (the paper's Table 3 queue sizes), every task compared."""
    cl = synth.make_cluster("pod")
    off, tasks = synth.make_tasks(2, cl.K, cl.M, cl.S, cl.B, 10, 100)
    ctx.load_cluster(cl)
    cmp.assert_tasks_equal(ctx.batch_tasks(off, tasks), _oracle_tasks(cl, off, tasks))


# ---- the paper's three-phase dispatcher (fs_dispatch) ------------------------------------------
def _oracle_dispatch(cl, reqs=None):
    return oracle.dispatch(cl.lat, cl.pow, cl.models, cl.states, cl.requests if reqs is None else reqs, 8)


def _mix_phases(cl, seed):
    """Push part of the requests into phase 2 (F_max retry), phase 3 (scale-out) and 'infeasible'."""
    u = synth.Stream(seed, "phases").uniform(cl.R)
    cl.requests["slo_ttft_ms"] = np.where(u < 0.3, cl.requests["slo_ttft_ms"] * 0.03, cl.requests["slo_ttft_ms"]).astype(np.float32)
    cl.requests["o_pred"] = np.where((u > 0.3) & (u < 0.4), 2 ** 20, cl.requests["o_pred"]).astype(np.uint32)   # fits no GPU's memory
    cl.requests["slo_tbt_ms"] = np.where(u > 0.95, 1e-3, cl.requests["slo_tbt_ms"]).astype(np.float32)


@pytest.mark.parametrize("seed", range(10))
def test_dispatch_ragged_dims_all_phases(ctx, seed):
    st = synth.Stream(seed, "ddims")
    K = int(st.randint(1, 1, 90)[0]); M = int(st.randint(1, 1, 9)[0])
    F = int(st.randint(1, 1, [64, 100][seed % 2])[0]); S = int(st.randint(1, 1, 20)[0]); B = int(st.randint(1, 1, 40)[0])
    cl = synth.make_custom(seed=1000 + seed, K=K, M=M, F=F, S=S, B=B, R=150, lo=1, hi=4)
    _mix_phases(cl, seed)
    if seed % 3 == 0:                                 # equal free memory everywhere: the SM_free / index tie-breakers
        cl.states["mem_free_mb"] = 30000.0
    ctx.load_cluster(cl)
    got = ctx.dispatch(cl.requests)
    cmp.assert_placement_equal(got, _oracle_dispatch(cl))


def test_dispatch_fig6(ctx):
    """Fig. 6 through the CUDA path: timestamps 150 / 180 / 210 against the SLO of 200, 45 J vs 30 J."""
    from test_oracle_dispatch import _toy, _gpu
    lat, pw, models, st, rq = _toy(K=3)
    for k, (t_avail, l, p) in enumerate([(100.0, 50.0, 900.0), (120.0, 60.0, 500.0), (150.0, 60.0, 100.0)]):
        _gpu(st, k, 1, 2, k, t_avail, 1e6)
        lat[0, 0, k, 1, 0] = l; pw[0, 0, k, 1, 0] = p
    ctx.load_profiles(lat, pw, np.ones(3, np.float32), models, synth.Params())
    ctx.set_gpu_state(st)
    o = ctx.dispatch(rq)[0]
    assert (o["gpu"], o["phi"], o["f_req"]) == (1, 1, 1) and o["energy_mj"] == np.float32(30000.0)


def test_dispatch_tie_heavy(ctx):
    cl = U.tie_heavy(synth.make_custom(seed=1020, K=40, M=3, F=12, S=6, B=5, R=96), 3)
    cl.states["mem_free_mb"] = np.round(cl.states["mem_free_mb"] / 10000.0) * 10000.0
    ctx.load_cluster(cl)
    cmp.assert_placement_equal(ctx.dispatch(cl.requests), _oracle_dispatch(cl))


def test_dispatch_full_size(ctx):
    """rack in full; pod at full size with a sample of requests recomputed by the oracle."""
    cl = synth.make_cluster("rack")
    ctx.load_cluster(cl)
    cmp.assert_placement_equal(ctx.dispatch(cl.requests), _oracle_dispatch(cl))
    cl = synth.make_cluster("pod")
    _mix_phases(cl, 5)
    ctx.load_cluster(cl)
    got = ctx.dispatch(cl.requests)
    idx = np.unique(synth.Stream(11, "sample").randint(2048, 0, cl.R - 1))
    cmp.assert_placement_equal(got[idx], _oracle_dispatch(cl, cl.requests[idx]))
    assert set(np.unique(got["f_req"]).tolist()) >= {1, 2, 3}


@pytest.mark.parametrize("R", [1, 19, 2959, 11840, 11841, 14799, 20000])
def test_request_counts_around_the_static_dynamic_boundary(ctx, R):
    """The scoring kernel hands requests to its warps by ticket (an atomic counter, two requests ahead); request counts
    around multiples of a full wave of warps (148 blocks x 20 warps = 2,960): every request exactly once at any R."""
    cl = synth.make_cluster("rack")
    reqs = synth.make_requests(4242 + R, R, cl.M)
    ctx.load_cluster(cl)
    got = ctx.place_batch(reqs)
    cmp.assert_placement_equal(got, oracle.place_batch(cl.lat, cl.pow, cl.models, cl.states, reqs, nthreads=16))


def test_device_requests_at_a_4_byte_aligned_address(ctx):
    """fs_request has 4-byte alignment: a device array that starts at any multiple of 4 must work
    (the scoring kernel prefetches requests with 16-byte asynchronous copies only when it can)."""
    import torch
    cl = synth.make_cluster("rack")
    ctx.load_cluster(cl)
    ref = ctx.place_batch(cl.requests)
    raw = torch.from_numpy(cl.requests.view(np.uint8).reshape(-1).copy())
    for off in (4, 8, 20):
        buf = torch.zeros(raw.numel() + 64, dtype=torch.uint8, device="cuda")
        buf[off:off + raw.numel()] = raw.cuda()
        out = torch.zeros(cl.R * 32 + 64, dtype=torch.uint8, device="cuda")
        ctx.place_batch(buf[off:], out=out[off:], R=cl.R)
        d = ctx.dispatch(buf[off:], out=torch.zeros(cl.R * 32, dtype=torch.uint8, device="cuda"), R=cl.R)
        torch.cuda.synchronize()
        assert out[off:off + cl.R * 32].cpu().numpy().tobytes() == ref.tobytes(), off


def test_host_pinned_async_equals_host(ctx):
    import paper_2606_30391_b200 as fs
    """FS_HOST_PINNED: page-locked host buffers, the call does not wait; same bytes as the blocking FS_HOST calls."""
    import torch
    cl = synth.make_cluster("rack")
    ctx.load_cluster(cl)
    ref_p = ctx.place_batch(cl.requests); ref_l = ctx.local_config(0); ref_d = ctx.dispatch(cl.requests)
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a).view(np.uint8).reshape(-1).copy()).pin_memory()
    h_st, h_rq = pin(cl.states), pin(cl.requests)
    h_p = torch.zeros(cl.R * 32, dtype=torch.uint8).pin_memory(); h_l = torch.zeros(cl.K * 48, dtype=torch.uint8).pin_memory()
    h_d = torch.zeros(cl.R * 32, dtype=torch.uint8).pin_memory()
    s = torch.cuda.Stream()
    ctx.set_gpu_state(h_st, stream=s, pinned=True)
    ctx.place_batch(h_rq, out=h_p, stream=s, pinned=True)
    ctx.local_config(0, n=cl.K, out=h_l, stream=s, pinned=True)
    rc = fs.lib().fs_dispatch(ctx._h, cl.R, h_rq.data_ptr(), h_d.data_ptr(), fs.FS_HOST_PINNED, s.cuda_stream)
    assert rc == 0
    s.synchronize()
    assert h_p.numpy().tobytes() == ref_p.tobytes() and h_l.numpy().tobytes() == ref_l.tobytes()
    assert h_d.numpy().tobytes() == ref_d.tobytes()
    # calls outside the serving loop reject the asynchronous space
    assert fs.lib().fs_ewr(ctx._h, 0, None, None, None, 0, None, None, fs.FS_HOST_PINNED, None) == -1


# ---- the sequential commit pass (fs_dispatch_commit, reading s34) -------------------------------------
def _assert_commit_equal(ctx, cl, reqs=None):
    reqs = cl.requests if reqs is None else reqs
    got, after = ctx.dispatch_commit(reqs)
    ref, st = oracle.dispatch_commit(cl.lat, cl.pow, cl.models, cl.states, reqs)
    cmp.assert_placement_equal(got, ref)
    for f in ("t_avail_ms", "mem_free_mb", "f_cur"):
        assert np.array_equal(after[f].view(np.uint32 if f != "f_cur" else np.int32),
                              st[f].view(np.uint32 if f != "f_cur" else np.int32)), f"after.{f}"
    return got


@pytest.mark.parametrize("seed", range(12))
def test_dispatch_commit_ragged_dims(ctx, seed):
    st = synth.Stream(seed, "cdims")
    K = int(st.randint(1, 1, [90, 2500][seed % 2])[0]); M = int(st.randint(1, 1, 9)[0])
    F = int(st.randint(1, 1, [64, 100][seed % 3 == 0])[0]); S = int(st.randint(1, 1, 20)[0]); B = int(st.randint(1, 1, 40)[0])
    cl = synth.make_custom(seed=1500 + seed, K=K, M=M, F=F, S=S, B=B, R=400, lo=1, hi=4)
    if seed % 4 == 1:
        cl.requests["slo_ttft_ms"] *= 0.1               # queues grow past the deadlines: phases 2 and 3
    if seed % 4 == 2:
        cl.states["mem_free_mb"] *= 0.01                # memory runs out during the batch
    if seed % 4 == 3:
        cl.states["mem_free_mb"] = 30000.0              # equal memory: the commit decides the tie-breaker
    ctx.load_cluster(cl)
    got = _assert_commit_equal(ctx, cl)
    snap = ctx.dispatch(cl.requests)
    assert got[0].tobytes() == snap[0].tobytes()
    # the context's own state is untouched: the snapshot dispatcher gives the same answers afterwards
    assert ctx.dispatch(cl.requests).tobytes() == snap.tobytes()


@pytest.mark.parametrize("K", [2049, 5000, 16384, 16385])
def test_dispatch_commit_many_gpus(ctx, K):
    """2,049 .. 16,384 GPUs: a thread-block cluster (minima through distributed shared memory); more: the
    single block with the records in global memory."""
    cl = synth.make_custom(seed=1600 + K % 97, K=K, M=6, F=20, S=8, B=12, R=300, lo=1, hi=4)
    u = synth.Stream(K, "cphase").uniform(cl.R)
    cl.requests["slo_ttft_ms"] = np.where(u < 0.3, cl.requests["slo_ttft_ms"] * 0.02, cl.requests["slo_ttft_ms"]).astype(np.float32)
    cl.requests["o_pred"] = np.where(u > 0.9, 2 ** 20, cl.requests["o_pred"]).astype(np.uint32)
    if K == 5000:
        cl.states["mem_free_mb"] = 30000.0              # every decision goes through the tie-breaker and the commit
    ctx.load_cluster(cl)
    got = _assert_commit_equal(ctx, cl)
    assert set(np.unique(got["f_req"]).tolist()) >= {1, 3}


def test_dispatch_commit_by_hand(ctx):
    """tests/test_oracle_commit.py::test_commit_by_hand through the CUDA path."""
    from test_oracle_dispatch import _toy, _gpu
    lat, pw, models, st, rq = _toy(K=2, F=2)
    rq = np.repeat(rq, 4); rq["o_pred"] = 20
    for k, t_avail in enumerate([10.0, 0.0]):
        _gpu(st, k, 1, 2, 0, t_avail, 1000.0)
    lat[0, 0, 0, 1, 0] = 50.0; lat[0, 1, 0, 1, 0] = 2.0; pw[0, :, 0, 1, 0] = 1.0
    lat[0, 0, 1, 1, 0] = 20.0; lat[0, 1, 1, 1, 0] = 1.0; pw[0, :, 1, 1, 0] = 9.0
    st["mem_free_mb"][1] = 500.0
    ctx.load_profiles(lat, pw, np.ones(2, np.float32), models, synth.Params())
    ctx.set_gpu_state(st)
    got, after = ctx.dispatch_commit(rq)
    assert got["gpu"].tolist() == [0, 0, 1, 1] and got["ttft_ms"].tolist() == [60.0, 152.0, 50.0, 142.0]
    assert after["t_avail_ms"].tolist() == [194.0, 184.0] and after["mem_free_mb"].tolist() == [956.0, 456.0]


def test_dispatch_commit_edges(ctx):
    import torch
    cl = synth.make_custom(seed=1530, K=33, M=3, F=7, S=5, B=4, R=64, lo=1, hi=4)
    ctx.load_cluster(cl)
    got, after = ctx.dispatch_commit(cl.requests[:0])      # R = 0: the records as polled
    assert len(got) == 0 and np.array_equal(after["t_avail_ms"], cl.states["t_avail_ms"])
    assert np.array_equal(after["f_cur"], cl.states["f_cur"])
    bad = cl.requests.copy(); bad["model"][5] = 99          # an invalid request is skipped, flagged on the next call
    got = np.zeros(cl.R, dtype=synth.PLACEMENT_DT); aft = np.zeros(cl.K, dtype=synth.GPU_AVAIL_DT)
    with pytest.raises(Exception):
        ctx.dispatch_commit(bad, out=got, after=aft)
    assert got["gpu"][5] == -1 and got["f_req"][5] == -1
    ok = cl.requests.copy(); ok = np.delete(ok, 5)
    ref, _ = oracle.dispatch_commit(cl.lat, cl.pow, cl.models, cl.states, ok)
    cmp.assert_placement_equal(np.delete(got, 5), ref)
    # device buffers
    dreq = torch.from_numpy(cl.requests.view(np.uint8)).cuda()
    dout = torch.zeros(cl.R * 32, dtype=torch.uint8, device="cuda"); daft = torch.zeros(cl.K * 16, dtype=torch.uint8, device="cuda")
    ctx.dispatch_commit(dreq, out=dout, after=daft, R=cl.R)
    torch.cuda.synchronize()
    ref, st = oracle.dispatch_commit(cl.lat, cl.pow, cl.models, cl.states, cl.requests)
    cmp.assert_placement_equal(dout.cpu().numpy().view(synth.PLACEMENT_DT), ref)
    assert np.array_equal(daft.cpu().numpy().view(synth.GPU_AVAIL_DT)["t_avail_ms"], st["t_avail_ms"])


def test_dispatch_commit_full_size(ctx):
    """rack in full; the pod's 1,024 GPUs with its first 8,192 requests (the oracle replays them serially)."""
    cl = synth.make_cluster("rack")
    ctx.load_cluster(cl)
    _assert_commit_equal(ctx, cl)
    cl = synth.make_cluster("pod")
    _mix_phases(cl, 5)
    ctx.load_cluster(cl)
    got = _assert_commit_equal(ctx, cl, cl.requests[:8192])
    assert set(np.unique(got["f_req"]).tolist()) >= {1, 2}


# ---- Algorithm 1 phase 1 (fs_llm_profiles) and the Energy Waste Ratio (fs_ewr) --------------------
def _assert_profiles_equal(got, ref):
    for f in ("sigma_p", "phi_p", "sigma_d", "phi_d", "need_units", "phi_l"):
        cmp._int_equal(got[f], ref[f], f"llm.{f}")
    for f in ("t_p_ms", "t_d_ms", "p_p_w", "p_d_w", "sm_units", "t_l_ms", "e_l_mj", "mem_mb"):
        cmp._float_close(got[f], ref[f], f"llm.{f}", True)


@pytest.mark.parametrize("seed", range(8))
def test_llm_profiles(ctx, seed):
    st = synth.Stream(seed, "ldims")
    M = int(st.randint(1, 1, 9)[0]); F = int(st.randint(1, 1, 70)[0]); S = int(st.randint(1, 1, 20)[0]); B = int(st.randint(1, 1, 40)[0])
    cl = synth.make_custom(seed=1200 + seed, K=2, M=M, F=F, S=S, B=B, R=0)
    if seed % 2:
        cl = U.tie_heavy(cl, seed)
    llms = synth.make_llms(seed, 300, cl.M)
    if seed % 4 == 1:
        llms["slo_ttft_ms"] *= 0.02; llms["slo_tbt_ms"] *= 0.2
    if seed % 4 == 2:
        llms["avg_in"][::3] = 0; llms["avg_out"][1::3] = 0
    ctx.load_cluster(cl)
    _assert_profiles_equal(ctx.llm_profiles(llms), oracle.llm_profile(cl.lat, cl.pow, cl.models, llms, 8))


def test_llm_profiles_pod_size(ctx):
    cl = synth.make_cluster("pod")
    llms = synth.make_llms(2, 4096, cl.M)
    ctx.load_cluster(cl)
    got = ctx.llm_profiles(llms)
    _assert_profiles_equal(got, oracle.llm_profile(cl.lat, cl.pow, cl.models, llms, 8))
    assert (got["phi_l"] >= 0).mean() > 0.9


def test_ewr(ctx):
    cl = synth.make_cluster("tiny")
    ctx.load_cluster(cl)
    st = synth.Stream(5, "ewr")
    for n, K in ((0, 3), (1, 1), (5000, 300), (70000, 4096)):
        g = st.randint(n, -1, K - 1).astype(np.int32); f = st.urange(n, 210, 1980).astype(np.float32)
        t = st.urange(n, 1, 1e4).astype(np.float32)
        fg, w, o, r = ctx.ewr(g, f, t, K)
        rfg, rw, ro, rr = oracle.ewr(g, f, t, K)
        assert np.array_equal(fg, rfg)
        # binary64 sums in a different (tree) order: 1e-12 relative
        assert abs(w - rw) <= 1e-12 * abs(rw) and abs(o - ro) <= 1e-12 * abs(ro) and abs(r - rr) <= 1e-12 * abs(rr)
    fg, w, o, r = ctx.ewr([0, 0, 1, -1], [1000, 1500, 1200, 900], [1, 2, 3, 4], 2)
    assert list(fg) == [1500.0, 1200.0] and w == 1500.0 ** 3 - 1000.0 ** 3 and r == w / o


# ---- Algorithm 1 phases 2-3 (fs_replace_plan) ------------------------------------------------------
@pytest.mark.parametrize("seed", range(10))
def test_replace_plan(ctx, seed):
    freq = np.linspace(210, 1980, [4, 16, 64][seed % 3]).astype(np.float32)
    S = [8, 16, 32][seed % 3]
    s_eff, m_eff = (S * 95) // 100, 76000.0
    n = [0, 1, 7, 33, 100, 257, 600, 64, 31, 1000][seed]
    l = synth.make_plan_llms(seed, n, S, freq)
    if seed % 4 == 3 and n:
        l["mem_mb"][::7] = 90000.0                  # exceed a whole GPU: stay unplaced
        l["need_units"][3::11] = s_eff + 1
    if seed == 4:
        l["f_mhz"] = freq[0]                        # all frequencies equal: index tie-breaks everywhere
    gpu_of, summ = ctx.replace_plan(l, s_eff, m_eff)
    rg, rs = oracle.replace_plan(l, s_eff, m_eff)
    assert summ == rs, (summ, rs)
    assert np.array_equal(gpu_of, rg)


def test_replace_plan_fig9(ctx):
    """The hand-built swap case of tests/test_oracle_plan.py through the CUDA path."""
    l = np.zeros(4, dtype=synth.PLAN_LLM_DT)
    l["need_units"] = 1; l["mem_mb"] = [30, 30, 30, 40]; l["f_mhz"] = [900, 1000, 1400, 1500]; l["t_ms"] = 10
    gpu_of, summ = ctx.replace_plan(l, 10, 100.0)
    assert list(gpu_of) == [1, 0, 0, 0] and summ == (1, 2, 2, 2)
    l["mem_mb"][3] = 50
    assert list(ctx.replace_plan(l, 10, 100.0)[0]) == [0, 0, 0, 1]


def test_replace_plan_from_profiles(ctx, fs):
    """Phase 1 feeds phases 2-3: profiles of 512 LLMs on the rack tables -> plan -> EWR, all on the GPU path."""
    cl = synth.make_cluster("rack")
    ctx.load_cluster(cl)
    llms = synth.make_llms(4, 512, cl.M)
    pr = ctx.llm_profiles(llms)
    ok = pr["phi_l"] >= 0
    pl = np.zeros(int(ok.sum()), dtype=synth.PLAN_LLM_DT)
    pl["need_units"] = pr["need_units"][ok]; pl["mem_mb"] = pr["mem_mb"][ok]
    pl["f_mhz"] = cl.freq_mhz[pr["phi_l"][ok]]; pl["t_ms"] = pr["t_l_ms"][ok]
    s_eff, m_eff = (cl.S * 95) // 100, 76000.0
    gpu_of, summ = ctx.replace_plan(pl, s_eff, m_eff)
    rg, rs = oracle.replace_plan(pl, s_eff, m_eff)
    assert summ == rs and np.array_equal(gpu_of, rg)
    fg, w, o, r = ctx.ewr(gpu_of, pl["f_mhz"], pl["t_ms"], summ[3])
    assert abs(r - oracle.ewr(gpu_of, pl["f_mhz"], pl["t_ms"], summ[3])[3]) <= 1e-12 * max(r, 1e-300)


# ---- Appendix E: transmission plan and selective migration ------------------------------------------
@pytest.mark.parametrize("n", [0, 1, 2, 7, 33, 120, 300])
def test_migration_plan(ctx, n):
    bytes_mb, bw, q = synth.make_migration(n, n, 10 * n)
    if n == 33:
        bw = np.round(bw / 25.0) * 25.0 + 25.0      # many equal costs: the tie rule decides the assignment
    dst, tot = ctx.migration_plan(bytes_mb, bw)
    rdst, rtot = oracle.assign(bytes_mb, bw)
    assert tot == rtot and np.array_equal(dst, rdst)
    assert sorted(dst) == list(range(n))            # a permutation whatever the tie-breaks
    flags, ms = ctx.migration_select(q)
    rflags, rms = oracle.migration_select(q)
    assert np.array_equal(flags, rflags) and np.array_equal(ms.view(np.uint32), rms.view(np.uint32))


def test_migration_plan_against_scipy(ctx):
    """The total is unique even where the assignment is not: check the CUDA path against a library solver."""
    from scipy.optimize import linear_sum_assignment
    bytes_mb, bw, _ = synth.make_migration(77, 64, 0)
    dst, tot = ctx.migration_plan(bytes_mb, bw)
    t = (bytes_mb[:, None] / bw).astype(np.float32)
    c = np.rint((t * np.float32(1000.0)).astype(np.float32)).astype(np.int64)
    rows, cols = linear_sum_assignment(c)
    assert tot == int(c[rows, cols].sum()) == int(c[np.arange(64), dst].sum())


# ---- the paper's largest cluster size (Table 3: 10,000 GPUs): GPUs split over several slices ---------
def test_ten_thousand_gpus_sampled(ctx):
    cl = synth.make_custom(seed=77, K=10000, M=32, F=64, S=16, B=64, R=3000, lo=1, hi=4)
    ctx.load_cluster(cl)
    got = ctx.place_batch(cl.requests)
    idx = np.unique(synth.Stream(13, "sample").randint(160, 0, cl.R - 1))
    cmp.assert_placement_equal(got[idx], _oracle_place(cl, cl.requests[idx]))
    one = ctx.place_batch(cl.requests[:1])            # a single arrival: the GPUs are split over the SMs
    cmp.assert_placement_equal(one, got[:1])
    dsp = ctx.dispatch(cl.requests)
    cmp.assert_placement_equal(dsp[idx], _oracle_dispatch(cl, cl.requests[idx]))
    # few arrivals: one block per request, its warps split the GPUs
    few = cl.requests[:150].copy()
    few["slo_ttft_ms"][::3] *= 0.03; few["o_pred"][1::5] = 2 ** 20; few["slo_tbt_ms"][2::7] = 1e-3
    got_few = ctx.dispatch(few)
    cmp.assert_placement_equal(got_few, _oracle_dispatch(cl, few))
    assert set(np.unique(got_few["f_req"]).tolist()) >= {1, 2, 3}
    cmp.assert_placement_equal(ctx.dispatch(few[:1]), got_few[:1])


# ---- extreme magnitudes: the pruning bounds and the early stop must stay sound -----------------------
@pytest.mark.parametrize("scale", [1e28, 1e-30, 1e-41])
def test_extreme_energy_scales(ctx, scale):
    """Power tables scaled so that energies sit near FLT_MAX, far below 1, and in the denormals."""
    cl = synth.make_custom(seed=1300, K=96, M=5, F=24, S=10, B=12, R=160, lo=1, hi=4)
    cl.pow = (cl.pow.astype(np.float64) * scale).astype(np.float32)
    cl.pow[cl.pow == 0] = np.float32(1e-45)                   # tables must stay > 0
    _check_all(ctx, cl, local=True, consol=True)
    cmp.assert_placement_equal(ctx.dispatch(cl.requests), _oracle_dispatch(cl))


def test_negative_and_huge_waits(ctx):
    cl = synth.make_custom(seed=1301, K=80, M=4, F=20, S=8, B=8, R=128, lo=1, hi=4)
    cl.states["t_avail_ms"][::3] = -500.0                      # a GPU that has been free for a while
    cl.states["t_avail_ms"][1::7] = 1e30
    cl.models["load_ms"][0] = 0.0
    cl.requests["slo_ttft_ms"][::5] = np.float32(np.inf)
    cl.requests["slo_tbt_ms"][::4] = np.float32(np.inf)
    _check_all(ctx, cl, local=False, consol=False)
    cmp.assert_placement_equal(ctx.dispatch(cl.requests), _oracle_dispatch(cl))


@pytest.mark.parametrize("S", [17, 24, 32])
def test_dense_scoring_up_to_32_shares(ctx, S):
    """The tiled scoring kernel covers every supported S (tiles of S rows per warp; fewer warps per block)."""
    for mode, (K, F) in enumerate([(300, 64), (2500, 33), (64, 17)]):
        cl = synth.make_custom(seed=1700 + S + mode, K=K, M=7, F=F, S=S, B=24, R=900, lo=1, hi=4)
        if mode == 1:
            cl.requests["slo_ttft_ms"] *= 3.0; cl.models["load_ms"] *= 0.1
        if mode == 2:
            cl = U.tie_heavy(cl, S)
        ctx.load_cluster(cl)
        ctx.set_work_stats(True)
        got = ctx.place_batch(cl.requests)
        stats = ctx.last_place_stats()
        ctx.set_work_stats(False)
        # counted only by the tiled kernel (the cold scan alone can be empty: another slice's result may prune it)
        assert stats["chunks_tested"] + stats["warm_pairs_tested"] > 0
        cmp.assert_placement_equal(got, oracle.place_batch(cl.lat, cl.pow, cl.models, cl.states, cl.requests, nthreads=16))


@pytest.mark.parametrize("F", [65, 96, 100, 128, 191, 256])
def test_dense_scoring_more_than_64_frequencies(ctx, F):
    """F > 64: the tiled kernel scores column blocks of 64 frequencies and merges them by key."""
    for mode, (K, S) in enumerate([(200, 16), (1500, 7), (40, 32)]):
        cl = synth.make_custom(seed=1800 + F + mode, K=K, M=6, F=F, S=S, B=20, R=500, lo=1, hi=4)
        if mode == 1:
            cl.requests["slo_ttft_ms"] *= 3.0; cl.models["load_ms"] *= 0.1
        if mode == 2:
            cl = U.tie_heavy(cl, F)
        ctx.load_cluster(cl)
        ctx.set_work_stats(True)
        got = ctx.place_batch(cl.requests)
        stats = ctx.last_place_stats()
        ctx.set_work_stats(False)
        assert stats["chunks_tested"] + stats["warm_pairs_tested"] > 0     # the tiled kernel ran
        ref = oracle.place_batch(cl.lat, cl.pow, cl.models, cl.states, cl.requests, nthreads=16)
        cmp.assert_placement_equal(got, ref)
        cmp.assert_placement_equal(ctx.place_batch(cl.requests), ref)        # the non-counting instantiation
        if F >= 128 and mode < 2:                             # winners beyond the first column block do occur
            assert (got["gpu"] >= 0).sum() > 50 and got["phi"].max() >= 64


# ---- randomised sweep: dims, load shapes and SLO regimes, every entry point of the hot path ----------
@pytest.mark.parametrize("block", range(4))
def test_random_clusters_all_entry_points(ctx, block):
    for seed in range(block * 30, block * 30 + 30):
        st = synth.Stream(seed, "fuzz")
        K = int(st.randint(1, 1, 400)[0]); M = int(st.randint(1, 1, 12)[0]); F = int(st.randint(1, 1, [64, 64, 160][seed % 3])[0])
        S = int(st.randint(1, 1, 32)[0]); B = int(st.randint(1, 1, 48)[0]); R = int(st.randint(1, 1, 700)[0])
        cl = synth.make_custom(seed=5000 + seed, K=K, M=M, F=F, S=S, B=B, R=R, lo=1, hi=4)
        mode = seed % 5
        if mode == 1:
            cl = U.tie_heavy(cl, seed)
        if mode == 2:                                   # many cold pairs can meet the TTFT deadline
            cl.requests["slo_ttft_ms"] *= 3.0; cl.models["load_ms"] *= 0.1
        if mode == 3:
            cl.requests["slo_ttft_ms"] *= 0.05
        if mode == 4:
            cl.states["mem_free_mb"] *= 0.02
        _check_all(ctx, cl)
        cmp.assert_placement_equal(ctx.dispatch(cl.requests), _oracle_dispatch(cl))


def test_fig8_step3_through_cuda(ctx):
    """Fig. 8 step 3 (tests/golden/fig8_step3.txt) through fs_local_config."""
    from test_oracle_pins import _fig8_cluster
    from test_golden import _rows
    rows = [[int(x) for x in r] for r in _rows("fig8_step3.txt")]
    cl = _fig8_cluster()
    ctx.load_profiles(cl.lat, cl.pow, np.array([r[0] for r in rows], np.float32), cl.models, synth.Params())
    ctx.set_gpu_state(cl.states)
    o = ctx.local_config(3 - 1)[0]                    # FS_OBJ_ENERGY | FS_SPLIT_MINSM
    chosen = min([r for r in rows if r[5]], key=lambda r: r[6])
    assert rows[int(o["phi"])][0] == chosen[0] == 1100
    assert tuple((int(s) + 1) * 10 for s in o["sigma"]) == tuple(chosen[1:5])
    assert o["energy_mj"] == np.float32(chosen[6] * 1000.0)
    for fl in ALL_FLAGS:
        cmp.assert_local_equal(ctx.local_config(fl), _oracle_local(cl, fl))


def test_step_is_capturable_into_a_cuda_graph(ctx):
    """The device-buffer calls are asynchronous and allocation-free after the first step: a whole step with the
    fork to a second stream and the join replays from one CUDA graph and gives the oracle's results."""
    import torch
    cl = synth.make_cluster("rack")
    dev = torch.device("cuda:0")
    tb = lambda a: torch.from_numpy(np.ascontiguousarray(a).view(np.uint8).reshape(-1)).to(dev)
    ctx.load_profiles(torch.from_numpy(cl.lat).to(dev), torch.from_numpy(cl.pow).to(dev), tb(cl.freq_mhz),
                      tb(cl.models), cl.params)
    ds, dr = tb(cl.states), tb(cl.requests)
    do = torch.empty(cl.R * 32, dtype=torch.uint8, device=dev)
    dl = torch.empty(cl.K * 48, dtype=torch.uint8, device=dev)
    side, ev0, ev1 = torch.cuda.Stream(), torch.cuda.Event(), torch.cuda.Event()

    def step(st):
        ctx.set_gpu_state(ds, stream=st)
        ev0.record(st); side.wait_event(ev0)
        ctx.local_config(0, n=cl.K, out=dl, stream=side)
        ctx.place_batch(dr, out=do, stream=st)
        ev1.record(side); st.wait_event(ev1)

    warm = torch.cuda.Stream()
    with torch.cuda.stream(warm):
        step(warm)                                      # first call at these sizes allocates scratch
    warm.synchronize()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g, stream=warm):
        step(torch.cuda.current_stream())
    do.zero_(); dl.zero_()
    g.replay(); g.replay()
    torch.cuda.synchronize()
    cmp.assert_placement_equal(do.cpu().numpy().view(synth.PLACEMENT_DT), _oracle_place(cl))
    cmp.assert_local_equal(dl.cpu().numpy().view(synth.LOCAL_CFG_DT), _oracle_local(cl, 0))
    # the next poll: other state records and other requests in the SAME device buffers, the same graph replayed.
    # fs_set_gpu_state is inside the graph, so the scan order and the per-model lists are rebuilt by the replay
    # (festina_eval.h: capture fs_set_gpu_state together with the placement calls that follow it)
    cl2 = synth.make_cluster("rack", seed=11)
    cl2.lat, cl2.pow, cl2.models = cl.lat, cl.pow, cl.models          # the tables stay those of the context
    cl2.states["t"]["mem_used_mb"][...] = 0                           # (mem_used is not read by these two calls)
    ds.copy_(tb(cl2.states)); dr.copy_(tb(cl2.requests))
    do.zero_(); dl.zero_()
    g.replay()
    torch.cuda.synchronize()
    cmp.assert_placement_equal(do.cpu().numpy().view(synth.PLACEMENT_DT), _oracle_place(cl2))
    cmp.assert_local_equal(dl.cpu().numpy().view(synth.LOCAL_CFG_DT), _oracle_local(cl2, 0))
    assert not np.array_equal(cl2.states["n_res"], cl.states["n_res"])


def test_first_call_of_a_size_inside_a_capture_is_refused_not_allocated(fs):
    """A call that would have to allocate (and wait for the device) while its stream is being captured returns
    FS_ERR_STATE and enqueues nothing, instead of invalidating the capture; after one call outside a capture the
    same call captures and replays."""
    import torch
    cl = synth.make_cluster("tiny")
    c = fs.Festina(0)
    c.load_cluster(cl)
    dev = torch.device("cuda", 0)
    d_reqs = torch.from_numpy(cl.requests.view(np.uint8).reshape(-1).copy()).to(dev)
    d_out = torch.zeros(cl.R * 32, dtype=torch.uint8, device=dev)
    torch.cuda.synchronize()
    s = torch.cuda.Stream()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.stream(s):
        g.capture_begin()
        try:
            with pytest.raises(fs.FestinaError) as e:
                c.place_batch(d_reqs, out=d_out, stream=s)          # first call with R requests: needs its buffers
            assert e.value.code == fs.FS_ERR_STATE
        finally:
            g.capture_end()
    torch.cuda.synchronize()
    c.place_batch(d_reqs, out=d_out, stream=s)                      # outside a capture: allocates
    torch.cuda.synchronize()
    g2 = torch.cuda.CUDAGraph()
    with torch.cuda.stream(s):
        g2.capture_begin()
        c.place_batch(d_reqs, out=d_out, stream=s)
        g2.capture_end()
    d_out.zero_()
    g2.replay()
    torch.cuda.synchronize()
    cmp.assert_placement_equal(d_out.cpu().numpy().view(synth.PLACEMENT_DT), _oracle_place(cl))
    c.close()


@pytest.mark.parametrize("variant", ["ties", "identical_gpus"])
def test_rack_tie_variants_full(ctx, variant):
    """configs[1] with tables quantised to a few powers of two and every SLO relaxed (ties inside a GPU), and with
    eight GPU records repeated (exact ties ACROSS GPUs: no bound is strict, every GPU of the best kind is swept);
    every tie must fall to the lowest flat index; compared in full."""
    cl = bench_work.make_variant("rack", variant)
    ctx.load_cluster(cl)
    cmp.assert_placement_equal(ctx.place_batch(cl.requests), _oracle_place(cl))


@pytest.mark.parametrize("variant", list(bench_work.VARIANTS))
def test_pod_workload_variants_sampled(ctx, variant):
    """configs[2] with a less degenerate shape: 4x the dynamic power (chosen frequencies spread over the levels)
    or cheap weight loads (cold starts meet the TTFT deadline, so the sorted cold scan does the work)."""
    cl = bench_work.make_variant("pod", variant)
    ctx.load_cluster(cl)
    got = ctx.place_batch(cl.requests)
    idx = np.arange(0, cl.R, 256 if variant in ("dynamic_power_x4", "cold_starts_feasible") else 1024)
    cmp.assert_placement_equal(got[idx], _oracle_place(cl, cl.requests[idx]))
    ok = got["gpu"] >= 0
    if variant == "dynamic_power_x4":
        assert np.bincount(got["phi"][ok]).max() / ok.sum() < 0.5
    cmp.assert_placement_equal(ctx.dispatch(cl.requests)[idx], _oracle_dispatch(cl, cl.requests[idx]))


# ---- the 64-bit argmin key: order of the fp32 -> u32 transform (SURVEY 8(c) "key encoding") --------------
def _key_order_cluster():
    """One request with no work of its own (L = 0, o_pred = 0: e_r = +0) against GPUs whose only tenant (another
    model, one prefill token, LAT 1 ms at phi 0 / 2 ms at phi 1 = F_curr, slack 1.5 ms so that only phi 0 is
    feasible) makes dE = fl(fl(A + 0) - Ecur) = fl(POW[phi 0] - 2 POW[phi 1]) take engineered values: the most
    negative finite floats, -1, negative subnormals, +0, positive subnormals, 1, huge, and -INF (Ecur overflows).
    The tenant's share selects the table row, so every GPU can have its own value."""
    tiny = np.float32(2.0 ** -149)
    rows = [(1.0, 1.5e38), (1.0, 5e29), (1.0, 1.0), (1e-40, 1e-40), (tiny, tiny), (2.0, 1.0),
            (3 * tiny, tiny), (3e-40, 1e-40), (3.0, 1.0), (3e30, 1.0), (3e38, 1e-3), (1.0, 3e38)]
    want = [-3e38 + 1, -1e30, -1.0, -1e-40, -float(tiny), 0.0, float(tiny), 1e-40, 1.0, 3e30, 3e38, -np.inf]
    M, F, S, B = 2, 2, 16, 1
    lat = np.ones((M, 2, F, S, B), dtype=np.float32)
    pw = np.ones_like(lat)
    lat[1, 0, 1] = 2.0
    for s, (p0, p1) in enumerate(rows):
        pw[1, 0, 0, s, 0], pw[1, 0, 1, s, 0] = p0, p1
    return lat, pw, rows, want


def test_argmin_key_orders_negative_zero_subnormal_huge_and_infinite_energies(ctx):
    lat, pw, rows, want = _key_order_cluster()
    n = len(rows)
    # GPU order scrambled against the value order; two copies of every row so that exact ties meet too
    order = [5, 0, 9, 3, 11, 7, 1, 10, 4, 8, 2, 6]
    tenants = lambda s: [dict(model=1, sigma=s, beta=(0, 0), q=(1, 0), slo=(1.5, 1e9))]
    full = U.mk_states([U.mk_state(f_cur=1, tenants=tenants(s)) for s in order + order])
    reqs = U.mk_requests([dict(model=0, L=0, o_pred=0)])
    by_value = sorted(range(n), key=lambda s: want[s])
    for drop in range(n):                               # remove the winners one by one: every adjacent pair of values meets
        states = full.copy()
        for s in by_value[:drop]:
            for k, sk in enumerate(order + order):
                if sk == s:
                    states[k]["n_res"] = 0
        cl = U.cluster_from(lat, pw, U.mk_models(2), states, reqs)
        ctx.load_cluster(cl)
        got = ctx.place_batch(cl.requests)
        ref = _oracle_place(cl, nthreads=1)
        cmp.assert_placement_equal(got, ref)
        # and against the value written above (not the oracle): the winner is the smallest remaining value, on
        # the FIRST of its two GPUs, share 0, phi 0
        s_win = by_value[drop]
        k_win = order.index(s_win)
        assert (int(got[0]["gpu"]), int(got[0]["sigma"]), int(got[0]["phi"])) == (k_win, 0, 0)
        with np.errstate(over="ignore"):
            e = np.float32(pw[1, 0, 0, s_win, 0]) - np.float32(2.0) * np.float32(pw[1, 0, 1, s_win, 0])
        assert got[0]["energy_mj"] == e
        assert np.isinf(e) or abs(float(e) - want[s_win]) <= 1e-6 * abs(want[s_win]) + 3e-45


def test_argmin_key_random_pairs(ctx):
    """Random pairs of energies of both signs and all magnitudes on two GPUs: the lower one wins, ties go to GPU 0."""
    st = synth.Stream(77, "keypairs")
    bits = st.randint(400, 0, 2 ** 31 - 1).astype(np.uint32)
    vals = bits.view(np.float32).copy()
    vals = vals[np.isfinite(vals) & (vals > 0)][:192]
    vals[::7] = vals[1::7][:len(vals[::7])]              # some exact duplicates
    M, F, B = 2, 2, 1
    for S in (8,):
        lat = np.ones((M, 2, F, S, B), dtype=np.float32)
        pw = np.ones_like(lat)
        lat[1, 0, 1] = 2.0
        reqs = U.mk_requests([dict(model=0, L=0, o_pred=0)])
        n_neg = 0
        for i in range(0, len(vals) - 3, 4):
            pw[1, 0, 0, 0, 0], pw[1, 0, 1, 0, 0] = vals[i], vals[i + 1]          # GPU 0's row
            pw[1, 0, 0, 1, 0], pw[1, 0, 1, 1, 0] = vals[i + 2], vals[i + 3]      # GPU 1's row
            states = U.mk_states([U.mk_state(f_cur=1, tenants=[dict(model=1, sigma=s, q=(1, 0), slo=(1.5, 1e9))])
                                  for s in (0, 1)])
            cl = U.cluster_from(lat, pw, U.mk_models(2), states, reqs)
            ctx.load_cluster(cl)
            got = ctx.place_batch(cl.requests)
            cmp.assert_placement_equal(got, _oracle_place(cl, nthreads=1))
            with np.errstate(over="ignore"):
                d = [np.float32(vals[i]) - np.float32(2.0) * np.float32(vals[i + 1]),
                     np.float32(vals[i + 2]) - np.float32(2.0) * np.float32(vals[i + 3])]
            assert int(got[0]["gpu"]) == (1 if d[1] < d[0] else 0)
            n_neg += int(min(d) < 0)
        assert n_neg > 5


# ---- the hand-computed pins of tests/test_oracle_pins.py through the CUDA path -----------------------------
def test_hand_computed_coupling_cases_through_cuda(ctx):
    import test_oracle_pins as pins
    for kw, want in ((dict(), (1, 0, -2280.0)), (dict(tenant0_tbt=11.0), (1, 1, 2820.0)), (dict(q1=0), (1, 0, 2100.0))):
        cl = pins._coupled_cluster(**kw)
        ctx.load_cluster(cl)
        o = ctx.place_batch(cl.requests)[0]
        assert (int(o["gpu"]), int(o["sigma"]), int(o["phi"])) == (0, want[0], want[1])
        assert o["energy_mj"] == np.float32(want[2])
    cl = pins._coupled_cluster(beta1=2)
    ctx.load_cluster(cl)
    assert ctx.place_batch(cl.requests)[0]["gpu"] == -1
    cl = pins._consol_busy_cluster()                    # pair score with busy destinations, by hand
    ctx.load_cluster(cl)
    out = ctx.consolidate()
    for a, (dst, phi, score, saving) in enumerate(pins.CONSOL_BY_HAND):
        assert (int(out[a]["dst"]), int(out[a]["phi"])) == (dst, phi), a
        assert out[a]["score_mj"] == np.float32(score) and out[a]["saving_mj"] == np.float32(saving), a
    cl = pins._power_cluster()
    ctx.load_cluster(cl)
    o = ctx.local_config(1 | 2)[0]
    assert (int(o["phi"]), int(o["sigma"][0]), tuple(o["beta"][0])) == (0, 1, (2, 0)) and o["cost"] == np.float32(102.0)
    assert o["energy_mj"] == np.float32(7276.0)
    o = ctx.local_config(0 | 2)[0]
    assert tuple(o["beta"][0]) == (1, 0) and o["cost"] == np.float32(7140.0) and o["power_w"] == np.float32(106.0)


# ---- fs_dispatch with no GPUs (every request scales out), fresh context and after a K > 0 state ------------
def test_dispatch_without_gpus_scales_out(fs):
    cl = synth.make_custom(seed=905, K=40, M=4, F=12, S=8, B=8, R=64, lo=1, hi=3)
    c = fs.Festina(0)                                   # fresh context: no warm lists were ever built
    c.load_profiles(cl.lat, cl.pow, cl.freq_mhz, cl.models, cl.params)
    c.set_gpu_state(cl.states[:0])
    got = c.dispatch(cl.requests)
    ref = oracle.dispatch(cl.lat, cl.pow, cl.models, cl.states[:0], cl.requests)
    cmp.assert_placement_equal(got, ref)
    assert (got["gpu"] == -1).all() and set(np.unique(got["f_req"])) <= {3, -1}
    c.set_gpu_state(cl.states)                          # K > 0, warm lists built ...
    cmp.assert_placement_equal(c.dispatch(cl.requests), oracle.dispatch(cl.lat, cl.pow, cl.models, cl.states, cl.requests))
    c.set_gpu_state(cl.states[:0])                      # ... and must not be read after K = 0
    got = c.dispatch(cl.requests)
    cmp.assert_placement_equal(got, ref)
    got2, after = c.dispatch_commit(cl.requests)
    assert (got2["gpu"] == -1).all() and len(after) == 0
    c.close()


# ---- the N > 1 result gather on an NCCL group (one rank: what a single GPU can exercise) ---------------------
def test_gather_records_on_an_nccl_group(tmp_path):
    """shard.gather_records with a CUDA byte tensor (the buffer a FS_DEVICE call wrote) on the nccl backend."""
    import subprocess
    import sys
    import textwrap
    import socket
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    sk = socket.socket(); sk.bind(("127.0.0.1", 0)); port = sk.getsockname()[1]; sk.close()
    code = textwrap.dedent(f"""
        import os, sys, numpy as np, torch, torch.distributed as dist
        sys.path.insert(0, {root!r})
        from paper_2606_30391_b200 import shard, synth
        import paper_2606_30391_b200 as fs
        os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT="{port}")
        torch.cuda.set_device(0)
        dist.init_process_group("nccl", rank=0, world_size=1, device_id=torch.device("cuda", 0))
        cl = synth.make_custom(seed=77, K=13, M=4, F=8, S=8, B=8, R=101, lo=1, hi=3)
        ctx = fs.Festina(0); ctx.load_cluster(cl)
        dev = torch.device("cuda", 0)
        d_req = torch.from_numpy(cl.requests.view(np.uint8).reshape(-1).copy()).to(dev)
        d_out = torch.empty(cl.R * 32, dtype=torch.uint8, device=dev)
        ctx.place_batch(d_req, out=d_out); torch.cuda.synchronize()
        full = shard.gather_records(d_out, [cl.R], dist, dtype=synth.PLACEMENT_DT)
        host = shard.gather_records(ctx.place_batch(cl.requests), [cl.R], dist)
        assert full.tobytes() == host.tobytes() == d_out.cpu().numpy().tobytes()
        dist.destroy_process_group(); print("gather ok")
    """)
    p = subprocess.run([sys.executable, "-c", code], capture_output=True, text=True, timeout=300)
    assert p.returncode == 0 and "gather ok" in p.stdout, (p.stdout + p.stderr)[-3000:]
