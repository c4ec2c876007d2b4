"""ctypes wrapper around the paper-model CPU oracle (oracle/sa_oracle_paper.cpp).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this.  It never imports the CUDA package.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from concurrent.futures import ThreadPoolExecutor
from typing import Iterable

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRCS = [os.path.join(_HERE, "sa_oracle_paper.cpp"), os.path.join(_HERE, "sa_oracle.cpp")]
_EXTRA = os.environ.get("ORACLE_CXXFLAGS", "").split()        # see oracle.py
_LIB = os.path.join(_HERE, "libsa_oracle_paper_san.so" if _EXTRA else "libsa_oracle_paper.so")
_lib = None


def build(force: bool = False) -> str:
    """g++ -O2: the paper-model oracle plus sa_oracle.cpp, whose Philox / mulhi / accept it links."""
    stale = (not os.path.exists(_LIB)) or any(os.path.getmtime(_LIB) < os.path.getmtime(s) for s in _SRCS)
    if force or stale:
        tmp = _LIB + ".tmp.%d" % os.getpid()
        subprocess.check_call(["g++", "-O2", "-std=c++17", "-shared", "-fPIC"] + _EXTRA + ["-o", tmp] + _SRCS)
        os.replace(tmp, _LIB)
    return _LIB


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        L.orcp_problem_create.restype = C.c_void_p
        L.orcp_problem_create.argtypes = [C.c_int, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.c_int,
                                          C.c_void_p, C.c_void_p]
        L.orcp_problem_destroy.argtypes = [C.c_void_p]
        L.orcp_objective.restype = C.c_uint32
        L.orcp_objective.argtypes = [C.c_void_p, C.c_void_p]
        L.orcp_simulate.restype = C.c_uint32
        L.orcp_simulate.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        L.orcp_objective_batch.argtypes = [C.c_void_p, C.c_void_p, C.c_int64, C.c_void_p]
        L.orcp_valid.restype = C.c_int
        L.orcp_valid.argtypes = [C.c_void_p, C.c_void_p]
        L.orcp_init_chain.argtypes = [C.c_void_p, C.c_uint64, C.c_uint32, C.c_int, C.c_void_p]
        L.orcp_propose.restype = C.c_int
        L.orcp_propose.argtypes = [C.c_void_p, C.c_uint32, C.c_uint32, C.c_void_p, C.c_int, C.c_void_p, C.c_void_p]
        L.orcp_domain_size.restype = C.c_int
        L.orcp_domain_size.argtypes = [C.c_void_p, C.c_int]
        L.orcp_domain_value.restype = C.c_int
        L.orcp_domain_value.argtypes = [C.c_void_p, C.c_int, C.c_int]
        L.orcp_run_chain.argtypes = [C.c_void_p, C.c_uint64, C.c_uint32, C.c_uint64, C.c_int64, C.c_int, C.c_int64,
                                     C.c_int, C.c_void_p, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p,
                                     C.c_void_p]
        _lib = L
    return _lib


def unpack_trace(rec: np.ndarray):
    rec = np.asarray(rec, dtype=np.uint64)
    return {
        "delta_cand": (rec & np.uint64(0xFFFFFFFF)).astype(np.uint32),
        "param": ((rec >> np.uint64(32)) & np.uint64(0xFFFFFF)).astype(np.int64),
        "code": ((rec >> np.uint64(56)) & np.uint64(0xF)).astype(np.int64),
        "accepted": ((rec >> np.uint64(60)) & np.uint64(1)).astype(bool),
        "new_best": ((rec >> np.uint64(61)) & np.uint64(1)).astype(bool),
        "null_move": ((rec >> np.uint64(62)) & np.uint64(1)).astype(bool),
    }


class PaperOracle:
    """The paper-model oracle bound to one problem (any object with the fields of problems.PaperProblem)."""

    def __init__(self, prob):
        self.prob = prob
        self._keep = [np.ascontiguousarray(prob.edge_src, dtype=np.int32),
                      np.ascontiguousarray(prob.edge_dst, dtype=np.int32),
                      np.ascontiguousarray(prob.fast, dtype=np.uint8),
                      np.ascontiguousarray(prob.init_state, dtype=np.uint8),
                      np.ascontiguousarray(prob.ref, dtype=np.uint8)]
        s, d, fa, ini, ref = self._keep
        self.N, self.E, self.K, self.T = prob.n_nodes, prob.n_edges, prob.n_cond, prob.n_steps
        self.P = 3 * self.E + 3 * self.N
        assert ini.shape == (self.K, self.N) and ref.shape == (self.K, self.T + 1, self.N)
        self.h = lib().orcp_problem_create(self.N, self.E, s.ctypes.data, d.ctypes.data, fa.ctypes.data, self.K, self.T,
                                           ini.ctypes.data, ref.ctypes.data)

    def __del__(self):
        try:
            if self.h:
                lib().orcp_problem_destroy(self.h)
                self.h = None
        except Exception:
            pass

    def _params(self, x) -> np.ndarray:
        x = np.ascontiguousarray(x, dtype=np.int8)
        assert x.shape[-1] == self.P, "parameter vector has the wrong length"
        return x

    def objective(self, params) -> int:
        return int(lib().orcp_objective(self.h, self._params(params).ctypes.data))

    fitness = objective

    def simulate(self, params) -> np.ndarray:
        """Whole time course uint8 [K][T+1][N] (t = 0 is the initial state)."""
        traj = np.zeros((self.K, self.T + 1, self.N), dtype=np.uint8)
        lib().orcp_simulate(self.h, self._params(params).ctypes.data, traj.ctypes.data)
        return traj

    def objective_batch(self, params, threads: int = 1) -> np.ndarray:
        x = self._params(params).reshape(-1, self.P)
        out = np.zeros(x.shape[0], dtype=np.uint32)
        if threads <= 1 or x.shape[0] < 2 * threads:
            lib().orcp_objective_batch(self.h, x.ctypes.data, x.shape[0], out.ctypes.data)
            return out
        bounds = np.linspace(0, x.shape[0], threads + 1).astype(np.int64)

        def work(t):
            a, b = int(bounds[t]), int(bounds[t + 1])
            if b > a:
                lib().orcp_objective_batch(self.h, x[a:b].ctypes.data, b - a, out[a:b].ctypes.data)
        with ThreadPoolExecutor(threads) as ex:
            list(ex.map(work, range(threads)))
        return out

    fitness_batch = objective_batch

    def valid(self, params) -> bool:
        return bool(lib().orcp_valid(self.h, self._params(params).ctypes.data))

    def domain(self, q: int):
        return [int(lib().orcp_domain_value(self.h, q, i)) for i in range(int(lib().orcp_domain_size(self.h, q)))]

    def init_chain(self, seed: int, chain: int, constrained: bool = False):
        x = np.zeros(self.P, dtype=np.int8)
        lib().orcp_init_chain(self.h, seed, chain, int(constrained), x.ctypes.data)
        return x, self.objective(x)

    def propose(self, x0: int, x1: int, cur, constrained: bool = False):
        """-> (parameter index, new value, moved)."""
        cur = self._params(cur)
        q, nv = C.c_int32(), C.c_int32()
        moved = lib().orcp_propose(self.h, x0, x1, cur.ctypes.data, int(constrained), C.byref(q), C.byref(nv))
        return q.value, nv.value, bool(moved)

    def run_chain(self, sched, chain: int, n_steps: int, g0: int = 0, state=None, trace: bool = True,
                  constrained: bool = False):
        if state is None:
            cur, f0 = self.init_chain(sched.seed, chain, constrained)
            best, fc, fb = cur.copy(), f0, f0
        else:
            cur, best, fc, fb = state
            cur = np.array(cur, dtype=np.int8)
            best = np.array(best, dtype=np.int8)
            f0 = None
        fcur, fbest = C.c_uint32(fc), C.c_uint32(fb)
        tr = np.zeros(n_steps if trace else 0, dtype=np.uint64)
        table = np.ascontiguousarray(sched.accept, dtype=np.uint32)
        lib().orcp_run_chain(self.h, sched.seed, chain, g0, n_steps, sched.n_levels, sched.steps_per_level, sched.dmax,
                             table.ctypes.data, int(constrained), cur.ctypes.data, best.ctypes.data, C.byref(fcur),
                             C.byref(fbest), tr.ctypes.data if trace else None)
        return {"cur": cur, "best": best, "fit_cur": fcur.value, "fit_best": fbest.value, "trace": tr, "init_fit": f0}

    def run_chains(self, sched, chains: Iterable[int], n_steps: int, threads: int = 1, trace: bool = True,
                   constrained: bool = False):
        chains = list(chains)
        if threads <= 1:
            return [self.run_chain(sched, c, n_steps, trace=trace, constrained=constrained) for c in chains]
        with ThreadPoolExecutor(threads) as ex:
            return list(ex.map(lambda c: self.run_chain(sched, c, n_steps, trace=trace, constrained=constrained), chains))


def simulate_fn(prob, params) -> np.ndarray:
    """The ``simulate`` callback problems.make_paper_problem expects, served by the oracle."""
    return PaperOracle(prob).simulate(params)


def run_levels(orc: "PaperOracle", sched, n_chains: int, n_levels: int, group_size: int = 0, g0: int = 0,
               states=None, threads: int = 1, constrained: bool = False):
    """PAPER.md Table 1 (:125-155) around the chain step, statement by statement (as oracle.run_levels):
    per level, n_iterations chain steps of every thread, then per group the smallest d_best (ties: the
    smallest chain) gives its x_best to every member as x_best and, at the top of the next level (:129),
    as x_current.  Returns the list of (cur, best, fit_cur, fit_best) after the last level."""
    R = n_chains
    group = R if group_size in (0, None) or group_size > R else group_size
    base = getattr(sched, "chain_id_base", 0)
    if states is None:
        states = []
        for c in range(R):
            x, f = orc.init_chain(sched.seed, base + c, constrained)
            states.append((x, x.copy(), f, f))
    g = g0
    assert g % sched.steps_per_level == 0, "levels start at level boundaries"
    for _ in range(n_levels):
        def advance(c):
            out = orc.run_chain(sched, base + c, sched.steps_per_level, g0=g, state=states[c], trace=False,
                                constrained=constrained)
            return (out["cur"], out["best"], out["fit_cur"], out["fit_best"])
        if threads > 1:
            with ThreadPoolExecutor(threads) as ex:
                states = list(ex.map(advance, range(R)))
        else:
            states = [advance(c) for c in range(R)]
        g += sched.steps_per_level
        for first in range(0, R, group):
            members = range(first, min(R, first + group))
            star = min(members, key=lambda c: (states[c][3], c))
            x_star, d_star = states[star][1], states[star][3]
            for c in members:
                states[c] = (x_star.copy(), x_star.copy(), d_star, d_star)
    return states
