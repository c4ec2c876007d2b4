"""Thin ctypes binding of libternary_sa.so — same names as include/ternary_sa.h, argument
marshalling only.  Every step of the path runs in the library's CUDA kernels; there is no CPU
fallback: importing this module raises if the library is missing.

PyTorch is plumbing: ``use_torch_plumbing()`` plugs its caching allocator in as the library's
device allocator and ``sa_create`` binds the handle to torch's current CUDA stream.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libternary_sa.so")

SA_OK, SA_EINVAL, SA_ENOMEM, SA_ECUDA = 0, -1, -2, -3
EXPORTS = ("sa_create", "sa_run", "sa_best", "sa_destroy", "sa_eval", "sa_simulate", "sa_get_chain",
           "sa_get_fitness", "sa_set_trace", "sa_get_trace", "sa_geometric_table", "sa_get_info",
           "sa_set_stream", "sa_set_allocator", "sa_int32_peak", "sa_imma_peak", "sa_last_error", "sa_plan_info",
           "sa_select_kernel", "sa_kernel_source_id", "sa_jit_check", "sa_run_levels", "sa_level_sync_static", "sa_clear_plan_cache", "sa_get_dense_info", "sa_get_level_stats",
           "sap_create", "sap_run", "sap_run_levels", "sap_best", "sap_destroy", "sap_eval", "sap_simulate",
           "sap_get_chain", "sap_get_fitness", "sap_set_trace", "sap_get_trace", "sap_get_level_stats", "sap_get_info",
           "sap_set_stream", "sap_jit_check")
SAP_CONSTRAINED, SAP_LEVEL_STATS = 1, 2
SA_KERNEL_AUTO, SA_KERNEL_GENERIC, SA_KERNEL_STATIC, SA_KERNEL_DENSE, SA_KERNEL_PAPER = 0, 1, 2, 3, 4
SA_CONSTRAINED, SA_LEVEL_STATS = 1, 2
SA_LEVEL_SYNC_STATIC_MAX_GROUPS = 65536

if not os.path.exists(LIB_PATH):
    raise ImportError(f"{LIB_PATH} is missing: run `python -m paper_2506_19866_b200.build` "
                      "(or __graft_entry__.build()); there is no CPU fallback")
_lib = C.CDLL(LIB_PATH)


class SaError(RuntimeError):
    def __init__(self, code: int, where: str):
        self.code = code
        msg = _lib.sa_last_error()
        super().__init__(f"{where} failed ({code}): {msg.decode() if msg else ''}")


class _Network(C.Structure):
    _fields_ = [("n_nodes", C.c_int32), ("n_edges", C.c_int32), ("edge_src", C.c_void_p), ("edge_dst", C.c_void_p),
                ("n_pairs", C.c_int32), ("th_lo", C.c_void_p), ("th_hi", C.c_void_p)]


class _Observations(C.Structure):
    _fields_ = [("n_cond", C.c_int32), ("n_steps", C.c_int32), ("n_obs", C.c_int32), ("obs_times", C.c_void_p),
                ("init_state", C.c_void_p), ("clamp", C.c_void_p), ("obs", C.c_void_p)]


class _Schedule(C.Structure):
    _fields_ = [("n_chains", C.c_int32), ("seed", C.c_uint64), ("n_levels", C.c_int32),
                ("steps_per_level", C.c_int32), ("dmax", C.c_int32), ("accept", C.c_void_p),
                ("chain_id_base", C.c_uint32), ("flags", C.c_uint32)]


ALLOC_FN = C.CFUNCTYPE(C.c_void_p, C.c_size_t, C.c_void_p)
FREE_FN = C.CFUNCTYPE(None, C.c_void_p)

_lib.sa_last_error.restype = C.c_char_p
_lib.sa_create.argtypes = [C.POINTER(_Network), C.POINTER(_Observations), C.POINTER(_Schedule), C.POINTER(C.c_void_p)]
_lib.sa_run.argtypes = [C.c_void_p, C.c_int64]
_lib.sa_run_levels.argtypes = [C.c_void_p, C.c_int64, C.c_int32]
_lib.sa_level_sync_static.argtypes = [C.c_void_p, C.c_int32]
_lib.sa_best.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
_lib.sa_destroy.argtypes = [C.c_void_p]
_lib.sa_destroy.restype = None
_lib.sa_eval.argtypes = [C.c_void_p, C.c_void_p, C.c_int64, C.c_void_p]
_lib.sa_simulate.argtypes = [C.POINTER(_Network), C.POINTER(_Observations), C.c_void_p, C.c_void_p]
_lib.sa_get_chain.argtypes = [C.c_void_p, C.c_int32, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
_lib.sa_get_fitness.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
_lib.sa_get_level_stats.argtypes = [C.c_void_p, C.c_void_p]
_lib.sa_set_trace.argtypes = [C.c_void_p, C.c_void_p, C.c_int32, C.c_int64]
_lib.sa_get_trace.argtypes = [C.c_void_p, C.c_void_p]
_lib.sa_geometric_table.argtypes = [C.c_double, C.c_double, C.c_int32, C.c_int32, C.c_void_p]
_lib.sa_get_info.argtypes = [C.c_void_p, C.c_void_p]
_lib.sa_get_dense_info.argtypes = [C.c_void_p, C.c_void_p]
_lib.sa_plan_info.argtypes = [C.POINTER(_Network), C.POINTER(_Observations), C.c_void_p]
_lib.sa_set_stream.argtypes = [C.c_void_p, C.c_void_p]
_lib.sa_set_allocator.argtypes = [C.c_void_p, C.c_void_p]
_lib.sa_int32_peak.argtypes = [C.c_void_p]
_lib.sa_imma_peak.argtypes = [C.c_void_p]
_lib.sa_select_kernel.argtypes = [C.c_void_p, C.c_int]
_lib.sa_jit_check.argtypes = [C.POINTER(_Network), C.POINTER(_Observations), C.c_int32, C.c_void_p, C.c_char_p, C.c_size_t]


class _PNetwork(C.Structure):
    _fields_ = [("n_nodes", C.c_int32), ("n_edges", C.c_int32), ("edge_src", C.c_void_p), ("edge_dst", C.c_void_p),
                ("fast", C.c_void_p)]


class _PObservations(C.Structure):
    _fields_ = [("n_cond", C.c_int32), ("n_steps", C.c_int32), ("init_state", C.c_void_p), ("ref", C.c_void_p)]


_lib.sap_create.argtypes = [C.POINTER(_PNetwork), C.POINTER(_PObservations), C.POINTER(_Schedule), C.c_uint32, C.POINTER(C.c_void_p)]
_lib.sap_run.argtypes = [C.c_void_p, C.c_int64]
_lib.sap_run_levels.argtypes = [C.c_void_p, C.c_int64, C.c_int32]
_lib.sap_best.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
_lib.sap_destroy.argtypes = [C.c_void_p]
_lib.sap_destroy.restype = None
_lib.sap_eval.argtypes = [C.c_void_p, C.c_void_p, C.c_int64, C.c_void_p]
_lib.sap_simulate.argtypes = [C.POINTER(_PNetwork), C.POINTER(_PObservations), C.c_void_p, C.c_void_p]
_lib.sap_get_chain.argtypes = [C.c_void_p, C.c_int32, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
_lib.sap_get_fitness.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
_lib.sap_set_trace.argtypes = [C.c_void_p, C.c_void_p, C.c_int32, C.c_int64]
_lib.sap_get_trace.argtypes = [C.c_void_p, C.c_void_p]
_lib.sap_get_level_stats.argtypes = [C.c_void_p, C.c_void_p]
_lib.sap_get_info.argtypes = [C.c_void_p, C.c_void_p]
_lib.sap_set_stream.argtypes = [C.c_void_p, C.c_void_p]
_lib.sap_jit_check.argtypes = [C.POINTER(_PNetwork), C.POINTER(_PObservations), C.c_void_p, C.c_char_p, C.c_size_t]


def _check(rc: int, where: str):
    if rc != SA_OK:
        raise SaError(rc, where)


def _arr(a, dtype) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=dtype)


def _marshal_problem(prob, need_obs: bool = True):
    keep = {
        "src": _arr(prob.edge_src, np.int32), "dst": _arr(prob.edge_dst, np.int32),
        "lo": _arr(prob.th_lo, np.int8), "hi": _arr(prob.th_hi, np.int8),
        "times": _arr(prob.obs_times, np.int32), "init": _arr(prob.init_state, np.uint8),
        "clamp": _arr(prob.clamp, np.uint8),
    }
    net = _Network(prob.n_nodes, prob.n_edges, keep["src"].ctypes.data, keep["dst"].ctypes.data,
                   keep["lo"].shape[0], keep["lo"].ctypes.data, keep["hi"].ctypes.data)
    obs_ptr = None
    if need_obs:
        keep["obs"] = _arr(prob.obs, np.uint8)
        obs_ptr = keep["obs"].ctypes.data
    obs = _Observations(prob.n_cond, prob.n_steps, keep["times"].shape[0], keep["times"].ctypes.data,
                        keep["init"].ctypes.data, keep["clamp"].ctypes.data, obs_ptr)
    return net, obs, keep


# ------------------------------------------------------------------------------- plumbing
_hooks = None


def use_torch_plumbing() -> None:
    """Device memory from PyTorch's CUDA caching allocator (process-wide hook)."""
    global _hooks
    if _hooks is not None:
        return
    import torch

    def _alloc(nbytes, stream):
        try:
            return torch.cuda.caching_allocator_alloc(int(nbytes), stream=int(stream or 0))
        except Exception:
            return None

    def _free(ptr):
        try:
            torch.cuda.caching_allocator_delete(int(ptr))
        except Exception:
            pass

    _hooks = (ALLOC_FN(_alloc), FREE_FN(_free))
    _check(_lib.sa_set_allocator(C.cast(_hooks[0], C.c_void_p), C.cast(_hooks[1], C.c_void_p)), "sa_set_allocator")


def sa_set_allocator_default() -> None:
    global _hooks
    _check(_lib.sa_set_allocator(None, None), "sa_set_allocator")
    _hooks = None


# ------------------------------------------------------------------------------- the ABI
def sa_geometric_table(t0: float, t_end: float, n_levels: int, dmax: int) -> np.ndarray:
    out = np.zeros((n_levels, dmax), dtype=np.uint32)
    _check(_lib.sa_geometric_table(t0, t_end, n_levels, dmax, out.ctypes.data), "sa_geometric_table")
    return out


def sa_create(prob, sched, stream: Optional[int] = None, flags: int = 0) -> int:
    """prob / sched: objects with the fields of problems.Problem / problems.Schedule.  Returns the handle."""
    net, obs, keep = _marshal_problem(prob)
    table = _arr(sched.accept, np.uint32)
    sc = _Schedule(sched.n_chains, sched.seed, sched.n_levels, sched.steps_per_level, sched.dmax,
                   table.ctypes.data, getattr(sched, "chain_id_base", 0), flags)
    h = C.c_void_p()
    _check(_lib.sa_create(C.byref(net), C.byref(obs), C.byref(sc), C.byref(h)), "sa_create")
    if stream is None and _hooks is not None:
        import torch
        stream = torch.cuda.current_stream().cuda_stream
    if stream:
        _check(_lib.sa_set_stream(h, C.c_void_p(stream)), "sa_set_stream")
    return h.value


def sa_set_stream(h: int, stream: int) -> None:
    _check(_lib.sa_set_stream(h, C.c_void_p(stream)), "sa_set_stream")


def sa_run(h: int, steps: int) -> None:
    _check(_lib.sa_run(h, steps), "sa_run")


def sa_run_levels(h: int, n_levels: int, group_size: int = 0) -> None:
    _check(_lib.sa_run_levels(h, n_levels, group_size), "sa_run_levels")


def sa_clear_plan_cache() -> None:
    _check(_lib.sa_clear_plan_cache(), "sa_clear_plan_cache")


def sa_level_sync_static(h: int, group_size: int = 0) -> None:
    """One level synchronisation with no device allocation (the winner table is a fixed array in the library,
    at most SA_LEVEL_SYNC_STATIC_MAX_GROUPS groups): for callers that cannot call cudaMalloc after set-up."""
    _check(_lib.sa_level_sync_static(h, group_size), "sa_level_sync_static")


def sa_best(h: int, n_params: int):
    fit, chain = C.c_uint32(), C.c_int32()
    params = np.zeros(n_params, dtype=np.int8)
    _check(_lib.sa_best(h, C.byref(fit), C.byref(chain), params.ctypes.data), "sa_best")
    return fit.value, chain.value, params


def sa_destroy(h: int) -> None:
    _lib.sa_destroy(h)


def sa_eval(h: int, params) -> np.ndarray:
    x = _arr(params, np.int8)
    x = x.reshape(-1, x.shape[-1])
    out = np.zeros(x.shape[0], dtype=np.uint32)
    _check(_lib.sa_eval(h, x.ctypes.data, x.shape[0], out.ctypes.data), "sa_eval")
    return out


def sa_simulate(prob, params) -> np.ndarray:
    net, obs, keep = _marshal_problem(prob, need_obs=False)
    x = _arr(params, np.int8)
    out = np.zeros((prob.n_cond, keep["times"].shape[0], prob.n_nodes), dtype=np.uint8)
    _check(_lib.sa_simulate(C.byref(net), C.byref(obs), x.ctypes.data, out.ctypes.data), "sa_simulate")
    return out


def sa_get_chain(h: int, chain: int, n_params: int):
    cur = np.zeros(n_params, dtype=np.int8)
    best = np.zeros(n_params, dtype=np.int8)
    fc, fb = C.c_uint32(), C.c_uint32()
    _check(_lib.sa_get_chain(h, chain, cur.ctypes.data, C.byref(fc), best.ctypes.data, C.byref(fb)), "sa_get_chain")
    return cur, fc.value, best, fb.value


def sa_get_fitness(h: int, n_chains: int):
    cur = np.zeros(n_chains, dtype=np.uint32)
    best = np.zeros(n_chains, dtype=np.uint32)
    _check(_lib.sa_get_fitness(h, cur.ctypes.data, best.ctypes.data), "sa_get_fitness")
    return cur, best


def sa_get_level_stats(h: int, n_levels: int) -> dict:
    out = np.zeros((n_levels, 4), dtype=np.uint64)
    _check(_lib.sa_get_level_stats(h, out.ctypes.data), "sa_get_level_stats")
    return {"steps": out[:, 0].astype(np.int64), "accepted": out[:, 1].astype(np.int64),
            "accepted_worse": out[:, 2].astype(np.int64), "improved": out[:, 3].astype(np.int64)}


def sa_set_trace(h: int, chains: Sequence[int], max_steps: int) -> None:
    c = _arr(list(chains), np.int32)
    _check(_lib.sa_set_trace(h, c.ctypes.data if c.size else None, int(c.size), max_steps), "sa_set_trace")


def sa_get_trace(h: int, n_chains: int, max_steps: int) -> np.ndarray:
    out = np.zeros((n_chains, max_steps), dtype=np.uint64)
    _check(_lib.sa_get_trace(h, out.ctypes.data), "sa_get_trace")
    return out


def sa_get_info(h: int) -> dict:
    info = np.zeros(16, dtype=np.int64)
    _check(_lib.sa_get_info(h, info.ctypes.data), "sa_get_info")
    keys = ("variant", "threads_per_cta", "chains_per_cta", "smem_bytes", "grid", "edge_slots", "sm_count", "launches",
            "passes", "edge_iterations", "rows", "split_nodes", "state_words_per_node", "state_entries",
            "static_regs", "team_warps")
    return dict(zip(keys, (int(v) for v in info)))


def sa_get_dense_info(h: int) -> dict:
    info = np.zeros(8, dtype=np.int64)
    _check(_lib.sa_get_dense_info(h, info.ctypes.data), "sa_get_dense_info")
    keys = ("applies", "row_tiles", "col_steps", "sparse", "team_warps", "ctas_per_sm", "slot_steps", "immas_per_step")
    return dict(zip(keys, (int(v) for v in info)))


def sa_plan_info(prob) -> dict:
    net, obs, keep = _marshal_problem(prob, need_obs=getattr(prob, "obs", None) is not None)
    info = np.zeros(16, dtype=np.int64)
    _check(_lib.sa_plan_info(C.byref(net), C.byref(obs), info.ctypes.data), "sa_plan_info")
    return {"variant": int(info[0]), "edge_slots": int(info[5]), "passes": int(info[8]), "edge_iterations": int(info[9]),
            "rows": int(info[10]), "split_nodes": int(info[11]), "state_words_per_node": int(info[12]),
            "state_entries": int(info[13]), "max_in_degree": int(info[14]), "clamped_mismatches": int(info[15])}


def sa_select_kernel(h: int, family: int) -> None:
    _check(_lib.sa_select_kernel(h, family), "sa_select_kernel")


def sa_kernel_source_id(family: int) -> str:
    """FNV-1a-64 (16 hex digits) of the run-time compiled source text the loaded library carries for a kernel family."""
    out = C.c_uint64()
    _check(_lib.sa_kernel_source_id(family, C.byref(out)), "sa_kernel_source_id")
    return f"{out.value:016x}"


def sa_jit_check(prob, n_chains: int) -> dict:
    """Host only: plan + NVRTC compile of the statically scheduled kernel for this problem."""
    net, obs, keep = _marshal_problem(prob, need_obs=getattr(prob, "obs", None) is not None)
    info = np.zeros(8, dtype=np.int64)
    log = C.create_string_buffer(16384)
    _check(_lib.sa_jit_check(C.byref(net), C.byref(obs), n_chains, info.ctypes.data, log, len(log)), "sa_jit_check")
    return {"applies": bool(info[0]), "team_warps": int(info[1]), "tiers": int(info[2]), "lane_slots": int(info[3]),
            "cubin_bytes": int(info[4]), "smem_bytes": int(info[5]), "dense_applies": bool(info[6]),
            "dense_cubin_bytes": int(info[7]), "log": log.value.decode(errors="replace")}


def sa_int32_peak() -> dict:
    out = np.zeros(6, dtype=np.float64)
    _check(_lib.sa_int32_peak(out.ctypes.data), "sa_int32_peak")
    return {"iadd3": out[0], "lop3": out[1], "imad": out[2], "mixed": out[3], "sm_count": int(out[4]), "sm_hz": out[5]}


def sa_imma_peak() -> dict:
    out = np.zeros(4, dtype=np.float64)
    _check(_lib.sa_imma_peak(out.ctypes.data), "sa_imma_peak")
    return {"imma_16832": out[0], "imma_sp_16864": out[1], "sm_count": int(out[2]), "sm_hz": out[3]}


def sa_last_error() -> str:
    msg = _lib.sa_last_error()
    return msg.decode() if msg else ""


# ------------------------------------------------------------------------------- the paper model
def _marshal_paper(prob, need_ref: bool = True):
    keep = {"src": _arr(prob.edge_src, np.int32), "dst": _arr(prob.edge_dst, np.int32), "fast": _arr(prob.fast, np.uint8),
            "init": _arr(prob.init_state, np.uint8)}
    net = _PNetwork(prob.n_nodes, prob.n_edges, keep["src"].ctypes.data, keep["dst"].ctypes.data, keep["fast"].ctypes.data)
    ref_ptr = None
    if need_ref:
        keep["ref"] = _arr(prob.ref, np.uint8)
        ref_ptr = keep["ref"].ctypes.data
    obs = _PObservations(prob.n_cond, prob.n_steps, keep["init"].ctypes.data, ref_ptr)
    return net, obs, keep


def sap_create(prob, sched, flags: int = 0, stream: Optional[int] = None) -> int:
    """prob / sched: objects with the fields of problems.PaperProblem / problems.Schedule.  Returns the handle."""
    net, obs, keep = _marshal_paper(prob)
    table = _arr(sched.accept, np.uint32)
    sc = _Schedule(sched.n_chains, sched.seed, sched.n_levels, sched.steps_per_level, sched.dmax,
                   table.ctypes.data, getattr(sched, "chain_id_base", 0), 0)
    h = C.c_void_p()
    _check(_lib.sap_create(C.byref(net), C.byref(obs), C.byref(sc), flags, C.byref(h)), "sap_create")
    if stream is None and _hooks is not None:
        import torch
        stream = torch.cuda.current_stream().cuda_stream
    if stream:
        _check(_lib.sap_set_stream(h, C.c_void_p(stream)), "sap_set_stream")
    return h.value


def sap_run(h: int, steps: int) -> None:
    _check(_lib.sap_run(h, steps), "sap_run")


def sap_run_levels(h: int, n_levels: int, group_size: int = 0) -> None:
    _check(_lib.sap_run_levels(h, n_levels, group_size), "sap_run_levels")


def sap_best(h: int, n_params: int):
    fit, chain = C.c_uint32(), C.c_int32()
    params = np.zeros(n_params, dtype=np.int8)
    _check(_lib.sap_best(h, C.byref(fit), C.byref(chain), params.ctypes.data), "sap_best")
    return fit.value, chain.value, params


def sap_destroy(h: int) -> None:
    _lib.sap_destroy(h)


def sap_eval(h: int, params) -> np.ndarray:
    x = _arr(params, np.int8)
    x = x.reshape(-1, x.shape[-1])
    out = np.zeros(x.shape[0], dtype=np.uint32)
    _check(_lib.sap_eval(h, x.ctypes.data, x.shape[0], out.ctypes.data), "sap_eval")
    return out


def sap_simulate(prob, params) -> np.ndarray:
    net, obs, keep = _marshal_paper(prob, need_ref=False)
    x = _arr(params, np.int8)
    out = np.zeros((prob.n_cond, prob.n_steps + 1, prob.n_nodes), dtype=np.uint8)
    _check(_lib.sap_simulate(C.byref(net), C.byref(obs), x.ctypes.data, out.ctypes.data), "sap_simulate")
    return out


def sap_get_chain(h: int, chain: int, n_params: int):
    cur = np.zeros(n_params, dtype=np.int8)
    best = np.zeros(n_params, dtype=np.int8)
    fc, fb = C.c_uint32(), C.c_uint32()
    _check(_lib.sap_get_chain(h, chain, cur.ctypes.data, C.byref(fc), best.ctypes.data, C.byref(fb)), "sap_get_chain")
    return cur, fc.value, best, fb.value


def sap_get_fitness(h: int, n_chains: int):
    cur = np.zeros(n_chains, dtype=np.uint32)
    best = np.zeros(n_chains, dtype=np.uint32)
    _check(_lib.sap_get_fitness(h, cur.ctypes.data, best.ctypes.data), "sap_get_fitness")
    return cur, best


def sap_set_trace(h: int, chains: Sequence[int], max_steps: int) -> None:
    c = _arr(list(chains), np.int32)
    _check(_lib.sap_set_trace(h, c.ctypes.data if c.size else None, int(c.size), max_steps), "sap_set_trace")


def sap_get_trace(h: int, n_chains: int, max_steps: int) -> np.ndarray:
    out = np.zeros((n_chains, max_steps), dtype=np.uint64)
    _check(_lib.sap_get_trace(h, out.ctypes.data), "sap_get_trace")
    return out


def sap_get_level_stats(h: int, n_levels: int) -> dict:
    out = np.zeros((n_levels, 4), dtype=np.uint64)
    _check(_lib.sap_get_level_stats(h, out.ctypes.data), "sap_get_level_stats")
    return {"steps": out[:, 0].astype(np.int64), "accepted": out[:, 1].astype(np.int64),
            "accepted_worse": out[:, 2].astype(np.int64), "improved": out[:, 3].astype(np.int64)}


def sap_get_info(h: int) -> dict:
    info = np.zeros(12, dtype=np.int64)
    _check(_lib.sap_get_info(h, info.ctypes.data), "sap_get_info")
    keys = ("lanes_per_chain", "node_slots", "edge_slots", "threads_per_cta", "chains_per_cta", "smem_bytes", "grid",
            "regs", "ctas_per_sm", "sm_count", "launches", "max_objective")
    return dict(zip(keys, (int(v) for v in info)))


def sap_jit_check(prob) -> dict:
    """Host only: plan + NVRTC compile of the paper-model kernels for this network."""
    net, obs, keep = _marshal_paper(prob, need_ref=getattr(prob, "ref", None) is not None)
    info = np.zeros(4, dtype=np.int64)
    log = C.create_string_buffer(16384)
    _check(_lib.sap_jit_check(C.byref(net), C.byref(obs), info.ctypes.data, log, len(log)), "sap_jit_check")
    return {"lanes_per_chain": int(info[0]), "node_slots": int(info[1]), "edge_slots": int(info[2]),
            "cubin_bytes": int(info[3]), "log": log.value.decode(errors="replace")}
