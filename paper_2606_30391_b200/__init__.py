"""paper_2606_30391_b200 — thin Python binding of libfestina_eval (the sm_100a CUDA library).

Argument marshalling only: every step of the hot path runs in the CUDA kernels behind the C ABI
declared in include/festina_eval.h.  There is no CPU fallback; importing the package without the
built library, or creating a context without a CUDA device, fails loudly.

Buffers may be numpy arrays (host; FS_HOST) or torch CUDA tensors (device; FS_DEVICE).  Record
layouts are the numpy dtypes of `paper_2606_30391_b200.synth` (mirrors of the C structs).
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import synth
from .build import LIB as _LIB_PATH, build as build_library

FS_OK, FS_ERR_ARG, FS_ERR_SHAPE, FS_ERR_STATE, FS_ERR_RANGE, FS_ERR_CUDA, FS_ERR_NOMEM = 0, -1, -2, -3, -4, -5, -6
FS_HOST, FS_DEVICE, FS_HOST_PINNED = 0, 1, 2
FS_OBJ_ENERGY, FS_OBJ_POWER, FS_SPLIT_EXHAUSTIVE, FS_SPLIT_MINSM = 0, 1, 0, 2

# every symbol include/festina_eval.h declares
SYMBOLS = ("fs_create", "fs_destroy", "fs_load_profiles", "fs_set_gpu_state", "fs_place_batch",
           "fs_local_config", "fs_consolidate", "fs_dispatch", "fs_dispatch_commit", "fs_batch_tasks", "fs_llm_profiles", "fs_ewr", "fs_replace_plan", "fs_replace_plan_static", "fs_migration_plan", "fs_migration_select", "fs_strerror", "fs_last_cuda_error",
           "fs_launch_count", "fs_set_work_stats", "fs_last_place_stats", "fs_set_timing", "fs_get_timing")
TIMERS = ("place_score", "place_decode", "summary", "local_slot", "local_split", "consol_agg",
          "consol_pair", "place_warm", "batch_tasks", "dispatch")


class FsDims(C.Structure):
    _fields_ = [("M", C.c_int32), ("F", C.c_int32), ("S", C.c_int32), ("B", C.c_int32)]


class FsParams(C.Structure):
    _fields_ = [("p_idle_w", C.c_float), ("horizon_ms", C.c_float), ("mem_cap_mb", C.c_float),
                ("delta_pct", C.c_int32)]


class FestinaError(RuntimeError):
    def __init__(self, code: int, where: str, cuda: int = 0):
        self.code = code
        msg = lib().fs_strerror(code).decode()
        super().__init__(f"{where}: {msg} (fs_status {code}" + (f", cudaError {cuda})" if cuda else ")"))


_lib = None


def lib() -> C.CDLL:
    """Load libfestina_eval.so (built in-tree by build.py).  Raises if it is missing."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(_LIB_PATH):
        raise ImportError(f"{_LIB_PATH} is not built: run `python -m paper_2606_30391_b200.build` "
                          "(or __graft_entry__.build()); there is no CPU fallback")
    L = C.CDLL(_LIB_PATH)
    vp, i32, u32 = C.c_void_p, C.c_int32, C.c_uint32
    L.fs_create.argtypes = [C.POINTER(vp), C.c_int]
    L.fs_destroy.argtypes = [vp]
    L.fs_load_profiles.argtypes = [vp, C.POINTER(FsDims), vp, vp, vp, vp, C.POINTER(FsParams), C.c_int, vp]
    L.fs_set_gpu_state.argtypes = [vp, i32, vp, C.c_int, vp]
    L.fs_place_batch.argtypes = [vp, i32, vp, vp, C.c_int, vp]
    L.fs_local_config.argtypes = [vp, i32, vp, u32, vp, C.c_int, vp]
    L.fs_consolidate.argtypes = [vp, vp, C.c_int, vp]
    L.fs_migration_plan.argtypes = [vp, i32, vp, vp, vp, vp, C.c_int, vp]
    L.fs_migration_select.argtypes = [vp, i32, vp, vp, vp, C.c_int, vp]
    L.fs_replace_plan.argtypes = [vp, i32, vp, i32, C.c_float, vp, vp, C.c_int, vp]
    L.fs_replace_plan_static.argtypes = [i32, vp, i32, C.c_float, vp, vp, vp]
    L.fs_llm_profiles.argtypes = [vp, i32, vp, vp, C.c_int, vp]
    L.fs_ewr.argtypes = [vp, i32, vp, vp, vp, i32, vp, vp, C.c_int, vp]
    L.fs_dispatch.argtypes = [vp, i32, vp, vp, C.c_int, vp]
    L.fs_dispatch_commit.argtypes = [vp, i32, vp, vp, vp, C.c_int, vp]
    L.fs_batch_tasks.argtypes = [vp, i32, vp, vp, vp, vp, i32, C.c_int, vp]
    L.fs_strerror.argtypes = [C.c_int]
    L.fs_strerror.restype = C.c_char_p
    L.fs_last_cuda_error.argtypes = [vp]
    L.fs_launch_count.argtypes = [vp]
    L.fs_launch_count.restype = C.c_uint64
    L.fs_set_work_stats.argtypes = [vp, C.c_int]
    L.fs_last_place_stats.argtypes = [vp, C.POINTER(C.c_uint64)]
    L.fs_set_timing.argtypes = [vp, C.c_int]
    L.fs_get_timing.argtypes = [vp, C.POINTER(C.c_float), C.c_int]
    for name in SYMBOLS:
        getattr(L, name)   # AttributeError if the library does not export it
    _lib = L
    return L


def _is_torch_cuda(x) -> bool:
    return hasattr(x, "is_cuda") and bool(x.is_cuda)


def _buf(x, nbytes: int | None = None):
    """(pointer, space, keepalive) of a numpy array, a torch tensor (CPU or CUDA) or None."""
    if x is None:
        return C.c_void_p(0), None, None
    if hasattr(x, "data_ptr"):                      # torch tensor
        assert x.is_contiguous()
        if nbytes is not None:
            assert x.numel() * x.element_size() >= nbytes, "buffer too small"
        return C.c_void_p(x.data_ptr()), (FS_DEVICE if x.is_cuda else FS_HOST), x
    a = np.ascontiguousarray(x)
    if nbytes is not None:
        assert a.nbytes >= nbytes, "buffer too small"
    return C.c_void_p(a.ctypes.data), FS_HOST, a


def _pin(sp, pinned: bool, *bufs):
    """FS_HOST -> FS_HOST_PINNED when the caller asks for the asynchronous page-locked host path."""
    if not pinned:
        return sp
    assert sp == FS_HOST, "pinned=True is for host buffers"
    for b in bufs:
        assert b is None or (hasattr(b, "is_pinned") and b.is_pinned()), "pinned=True needs page-locked torch tensors"
    return FS_HOST_PINNED


def _stream_ptr(stream) -> C.c_void_p:
    if stream is None:
        return C.c_void_p(0)
    if hasattr(stream, "cuda_stream"):
        return C.c_void_p(stream.cuda_stream)
    return C.c_void_p(int(stream))


FS_PLAN_STATIC_MAX_N = 1024   # festina_eval.h


def replace_plan_static(llms, s_eff: int, m_eff: float, gpu_of, summary, stream=None) -> None:
    """fs_replace_plan_static: Algorithm 1 phases 2-3 without a context and without any allocation.

    For a process that cannot (HBM already handed to a serving engine) or must not (cudaMalloc / cudaFree
    stall the inference streams it shares the GPU with) allocate device memory when it needs a plan.
    `llms` (n fs_plan_llm records, 16 bytes each), `gpu_of` (n int32) and `summary` (4 int32) are torch CUDA
    tensors of the caller, on the current device; nothing is copied, the kernel is enqueued on `stream` and
    the results are valid once that stream has been synchronised.  At most FS_PLAN_STATIC_MAX_N LLMs: the
    working arrays are a fixed array inside the library, shared by all calls (do not overlap two calls on
    one GPU).  Raises FestinaError (FS_ERR_SHAPE) beyond that limit."""
    for t in (llms, gpu_of, summary):
        assert _is_torch_cuda(t) and t.is_contiguous(), "device tensors only: this path copies nothing"
    n = llms.numel() * llms.element_size() // 16
    assert gpu_of.numel() * gpu_of.element_size() >= 4 * n and summary.numel() * summary.element_size() >= 16
    rc = lib().fs_replace_plan_static(n, C.c_void_p(llms.data_ptr()), int(s_eff), float(m_eff),
                                      C.c_void_p(gpu_of.data_ptr()), C.c_void_p(summary.data_ptr()), _stream_ptr(stream))
    if rc != FS_OK:
        where = "fs_replace_plan_static"
        if rc == FS_ERR_SHAPE:
            where += f" (n = {n} LLMs, the built-in scratch array holds at most {FS_PLAN_STATIC_MAX_N})"
        raise FestinaError(rc, where)


class Festina:
    """One libfestina_eval context on one CUDA device (not thread-safe, see festina_eval.h)."""

    def __init__(self, device: int = 0):
        self._h = C.c_void_p(0)
        rc = lib().fs_create(C.byref(self._h), int(device))
        if rc != FS_OK:
            self._h = C.c_void_p(0)
            raise FestinaError(rc, "fs_create")
        self.device = device
        self.dims = None
        self.K = 0

    def close(self):
        if self._h:
            lib().fs_destroy(self._h)
            self._h = C.c_void_p(0)

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _check(self, rc: int, where: str):
        if rc != FS_OK:
            raise FestinaError(rc, where, lib().fs_last_cuda_error(self._h))

    # -- the five calls of the boundary ----------------------------------------------------
    def load_profiles(self, lat, pow_, freq_mhz, models, params: synth.Params, stream=None):
        M, P, F, S, B = tuple(lat.shape)
        assert P == 2 and tuple(pow_.shape) == tuple(lat.shape)
        n = M * 2 * F * S * B * 4
        pl, sp, k1 = _buf(lat, n)
        pp, sp2, k2 = _buf(pow_, n)
        pf, sp3, k3 = _buf(freq_mhz, F * 4)
        pm, sp4, k4 = _buf(models, M * 16)
        assert sp == sp2 == sp3 == sp4, "all bulk pointers of one call live in one memory space"
        dims = FsDims(M, F, S, B)
        prm = FsParams(params.p_idle_w, params.horizon_ms, params.mem_cap_mb, params.delta_pct)
        rc = lib().fs_load_profiles(self._h, C.byref(dims), pl, pp, pf, pm, C.byref(prm), sp,
                                    _stream_ptr(stream))
        self._check(rc, "fs_load_profiles")
        self.dims = (M, F, S, B)
        self.K = 0

    def set_gpu_state(self, states, K: int | None = None, stream=None, pinned: bool = False):
        if K is None:
            K = len(states) if not hasattr(states, "data_ptr") else states.numel() * states.element_size() // 128
        ps, sp, keep = _buf(states, K * 128)
        sp = _pin(sp if sp is not None else FS_HOST, pinned, states)
        rc = lib().fs_set_gpu_state(self._h, K, ps, sp, _stream_ptr(stream))
        self._check(rc, "fs_set_gpu_state")
        self.K = K

    def place_batch(self, reqs, out=None, R: int | None = None, stream=None, pinned: bool = False):
        """Returns a numpy record array (host inputs) or writes into `out` (device tensors).  pinned=True:
        page-locked host tensors, asynchronous (FS_HOST_PINNED): synchronise `stream` before reading `out`."""
        if R is None:
            R = len(reqs) if not hasattr(reqs, "data_ptr") else reqs.numel() * reqs.element_size() // 32
        pr, sp, keep = _buf(reqs, R * 32)
        if sp is None:
            sp = FS_HOST
        if out is None:
            assert sp == FS_HOST, "device inputs need a device `out` tensor"
            out = np.zeros(R, dtype=synth.PLACEMENT_DT)
        po, spo, keep2 = _buf(out, R * 32)
        assert spo == sp or R == 0
        sp = _pin(sp, pinned, reqs, out)
        rc = lib().fs_place_batch(self._h, R, pr, po, sp, _stream_ptr(stream))
        self._check(rc, "fs_place_batch")
        return out

    def dispatch(self, reqs, out=None, R: int | None = None, stream=None):
        """fs_dispatch: the paper's three-phase dispatcher at (F_curr, SM_free)."""
        if R is None:
            R = len(reqs) if not hasattr(reqs, "data_ptr") else reqs.numel() * reqs.element_size() // 32
        pr, sp, keep = _buf(reqs, R * 32)
        if sp is None:
            sp = FS_HOST
        if out is None:
            assert sp == FS_HOST, "device inputs need a device `out` tensor"
            out = np.zeros(R, dtype=synth.PLACEMENT_DT)
        po, spo, keep2 = _buf(out, R * 32)
        assert spo == sp or R == 0
        self._check(lib().fs_dispatch(self._h, R, pr, po, sp, _stream_ptr(stream)), "fs_dispatch")
        return out

    def dispatch_commit(self, reqs, out=None, after=None, R: int | None = None, stream=None):
        """fs_dispatch_commit: the dispatcher with the sequential commit pass; returns (placements, the
        (T_avail, free memory, F_curr) records after the last commit)."""
        if R is None:
            R = len(reqs) if not hasattr(reqs, "data_ptr") else reqs.numel() * reqs.element_size() // 32
        pr, sp, keep = _buf(reqs, R * 32)
        if sp is None:
            sp = FS_HOST
        if out is None:
            assert sp == FS_HOST, "device inputs need device `out` / `after` tensors"
            out = np.zeros(R, dtype=synth.PLACEMENT_DT)
            after = np.zeros(self.K, dtype=synth.GPU_AVAIL_DT)
        po, spo, keep2 = _buf(out, R * 32)
        pa, spa, keep3 = _buf(after, self.K * 16)
        assert (spo == sp or R == 0) and spa in (None, sp)
        self._check(lib().fs_dispatch_commit(self._h, R, pr, po, pa, sp, _stream_ptr(stream)), "fs_dispatch_commit")
        return out, after

    def local_config(self, flags: int = 0, gpu_ids=None, n: int | None = None, out=None, stream=None, pinned: bool = False):
        if gpu_ids is not None and not hasattr(gpu_ids, "data_ptr"):
            gpu_ids = np.ascontiguousarray(gpu_ids, dtype=np.int32)
        if n is None:
            n = self.K if gpu_ids is None else (len(gpu_ids) if not hasattr(gpu_ids, "data_ptr") else gpu_ids.numel())
        pi, spi, keep = _buf(gpu_ids)
        if out is None:
            assert spi in (None, FS_HOST)
            out = np.zeros(n, dtype=synth.LOCAL_CFG_DT)
        po, spo, keep2 = _buf(out, n * 48)
        assert spi is None or spi == spo
        spo = _pin(spo, pinned, gpu_ids, out)
        rc = lib().fs_local_config(self._h, n, pi, flags, po, spo, _stream_ptr(stream))
        self._check(rc, "fs_local_config")
        return out

    def batch_tasks(self, task_off, tasks, gpu_ids=None, out=None, n: int | None = None,
                    n_tasks: int | None = None, stream=None):
        """fs_batch_tasks: priority score + batching with bypass for n GPUs (host arrays or device tensors)."""
        host = not hasattr(tasks, "data_ptr")
        if host:
            task_off = np.ascontiguousarray(task_off, dtype=np.int32)
            tasks = np.ascontiguousarray(tasks)
            if gpu_ids is not None:
                gpu_ids = np.ascontiguousarray(gpu_ids, dtype=np.int32)
            n = len(task_off) - 1 if n is None else n
            n_tasks = len(tasks) if n_tasks is None else n_tasks
            if out is None:
                out = np.zeros(n_tasks, dtype=synth.TASK_OUT_DT)
        else:
            assert out is not None and n is not None and n_tasks is not None
        pi, _, k0 = _buf(gpu_ids)
        pf, spf, k1 = _buf(task_off)
        pt, spt, k2 = _buf(tasks, n_tasks * 24)
        po, spo, k3 = _buf(out, n_tasks * 16)
        sp = spf if spf is not None else FS_HOST
        rc = lib().fs_batch_tasks(self._h, n, pi, pf, pt, po, n_tasks, sp, _stream_ptr(stream))
        self._check(rc, "fs_batch_tasks")
        return out

    def llm_profiles(self, llms, out=None, n: int | None = None, stream=None):
        """fs_llm_profiles: Algorithm 1 phase 1 per active LLM (host arrays or device tensors)."""
        if n is None:
            n = len(llms) if not hasattr(llms, "data_ptr") else llms.numel() * llms.element_size() // 32
        pi, sp, keep = _buf(llms, n * 32)
        if sp is None:
            sp = FS_HOST
        if out is None:
            assert sp == FS_HOST
            out = np.zeros(n, dtype=synth.LLM_PROFILE_DT)
        po, spo, keep2 = _buf(out, n * 48)
        self._check(lib().fs_llm_profiles(self._h, n, pi, po, sp, _stream_ptr(stream)), "fs_llm_profiles")
        return out

    def ewr(self, gpu_of, f_mhz, t_ms, K: int, stream=None):
        """fs_ewr on host arrays: returns (F_g [K], E_waste, E_optimal, EWR)."""
        gpu_of = np.ascontiguousarray(gpu_of, dtype=np.int32)
        f_mhz = np.ascontiguousarray(f_mhz, dtype=np.float32)
        t_ms = np.ascontiguousarray(t_ms, dtype=np.float32)
        fg = np.zeros(max(K, 1), dtype=np.float32)
        out = np.zeros(3, dtype=np.float64)
        p = lambda a: C.c_void_p(a.ctypes.data)
        rc = lib().fs_ewr(self._h, len(gpu_of), p(gpu_of), p(f_mhz), p(t_ms), K, p(fg), p(out), FS_HOST,
                          _stream_ptr(stream))
        self._check(rc, "fs_ewr")
        return fg[:K], float(out[0]), float(out[1]), float(out[2])

    def replace_plan(self, llms, s_eff: int, m_eff: float, stream=None):
        """fs_replace_plan on host arrays: returns (gpu_of [n], (N_sm, N_mem, N_min, N_active))."""
        llms = np.ascontiguousarray(llms)
        gpu_of = np.full(max(len(llms), 1), -1, dtype=np.int32)
        summ = np.zeros(4, dtype=np.int32)
        p = lambda a: C.c_void_p(a.ctypes.data)
        rc = lib().fs_replace_plan(self._h, len(llms), p(llms) if len(llms) else C.c_void_p(0), s_eff, m_eff,
                                   p(gpu_of), p(summ), FS_HOST, _stream_ptr(stream))
        self._check(rc, "fs_replace_plan")
        return gpu_of[:len(llms)], tuple(int(x) for x in summ)

    def migration_plan(self, bytes_mb, bw_mb_per_ms, stream=None):
        """fs_migration_plan on host arrays: returns (dst_of [n], total cost in microseconds)."""
        bytes_mb = np.ascontiguousarray(bytes_mb, dtype=np.float32)
        bw = np.ascontiguousarray(bw_mb_per_ms, dtype=np.float32)
        n = len(bytes_mb)
        dst = np.full(max(n, 1), -1, dtype=np.int32)
        tot = np.zeros(1, dtype=np.int64)
        p = lambda a: C.c_void_p(a.ctypes.data)
        rc = lib().fs_migration_plan(self._h, n, p(bytes_mb), p(bw), p(dst), p(tot), FS_HOST, _stream_ptr(stream))
        self._check(rc, "fs_migration_plan")
        return dst[:n], int(tot[0])

    def migration_select(self, reqs, stream=None):
        """fs_migration_select on host arrays: returns (flags u8, migration time ms)."""
        reqs = np.ascontiguousarray(reqs)
        r = len(reqs)
        flags = np.zeros(max(r, 1), dtype=np.uint8)
        ms = np.zeros(max(r, 1), dtype=np.float32)
        p = lambda a: C.c_void_p(a.ctypes.data)
        rc = lib().fs_migration_select(self._h, r, p(reqs), p(flags), p(ms), FS_HOST, _stream_ptr(stream))
        self._check(rc, "fs_migration_select")
        return flags[:r], ms[:r]

    def consolidate(self, out=None, stream=None, pinned: bool = False):
        if out is None:
            out = np.zeros(self.K, dtype=synth.CONSOL_DT)
        po, spo, keep = _buf(out, self.K * 16)
        spo = _pin(spo, pinned, out)
        rc = lib().fs_consolidate(self._h, po, spo, _stream_ptr(stream))
        self._check(rc, "fs_consolidate")
        return out

    # -- diagnostics -------------------------------------------------------------------------
    @property
    def launch_count(self) -> int:
        return int(lib().fs_launch_count(self._h))

    def set_work_stats(self, on: bool = True):
        self._check(lib().fs_set_work_stats(self._h, int(on)), "fs_set_work_stats")

    def last_place_stats(self) -> dict:
        """Work counters of the last fs_place_batch run with set_work_stats(True) (festina_eval.h)."""
        names = ("chunks_tested", "cold_pairs_eligible", "cold_pairs_swept", "cold_candidates_swept",
                 "warm_pairs_tested", "pairs_scored", "candidates_scored", "requests", "tiles_built")
        o = (C.c_uint64 * len(names))()                  # FS_NSTATS
        self._check(lib().fs_last_place_stats(self._h, o), "fs_last_place_stats")
        return {n: int(o[i]) for i, n in enumerate(names)}

    def set_timing(self, on: bool = True):
        self._check(lib().fs_set_timing(self._h, int(on)), "fs_set_timing")

    def get_timing(self) -> dict:
        """Device time in ms of the most recent launch of each timed kernel (see fs_timer)."""
        ms = (C.c_float * len(TIMERS))()
        self._check(lib().fs_get_timing(self._h, ms, len(TIMERS)), "fs_get_timing")
        return {k: float(ms[i]) for i, k in enumerate(TIMERS) if ms[i] >= 0}

    def load_cluster(self, cl: synth.Cluster, stream=None):
        """Convenience: fs_load_profiles + fs_set_gpu_state from a synthetic cluster (host)."""
        self.load_profiles(cl.lat, cl.pow, cl.freq_mhz, cl.models, cl.params, stream)
        self.set_gpu_state(cl.states, stream=stream)
        return self
