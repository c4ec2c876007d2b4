"""ctypes wrapper around the CPU oracle (oracle/sa_oracle.cpp).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this.  It never imports the CUDA package.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from concurrent.futures import ThreadPoolExecutor
from typing import Iterable, List, Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "sa_oracle.cpp")
# ORACLE_CXXFLAGS="-fsanitize=address,undefined -g": an instrumented copy of the oracle for the pin tests
# (run them with LD_PRELOAD=$(g++ -print-file-name=libasan.so)); it is built beside the plain one
_EXTRA = os.environ.get("ORACLE_CXXFLAGS", "").split()
_LIB = os.path.join(_HERE, "libsa_oracle_san.so" if _EXTRA else "libsa_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile the oracle with g++ -O2 (single-threaded C++, no SIMD flags)."""
    stale = (not os.path.exists(_LIB)) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC)
    if force or stale:
        tmp = _LIB + ".tmp.%d" % os.getpid()
        subprocess.check_call(["g++", "-O2", "-std=c++17", "-shared", "-fPIC"] + _EXTRA + ["-o", tmp, _SRC])
        os.replace(tmp, _LIB)
    return _LIB


def _ptr(a: np.ndarray, ct):
    return a.ctypes.data_as(C.POINTER(ct))


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        L.orc_problem_create.restype = C.c_void_p
        L.orc_problem_create.argtypes = [C.c_int, C.c_int, C.c_void_p, C.c_void_p, C.c_int, C.c_void_p,
                                         C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_void_p, C.c_void_p,
                                         C.c_void_p, C.c_void_p]
        L.orc_problem_destroy.argtypes = [C.c_void_p]
        L.orc_fitness.restype = C.c_uint32
        L.orc_fitness.argtypes = [C.c_void_p, C.c_void_p]
        L.orc_simulate.restype = C.c_uint32
        L.orc_simulate.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        L.orc_fitness_batch.argtypes = [C.c_void_p, C.c_void_p, C.c_int64, C.c_void_p]
        L.orc_philox4x32_10.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        L.orc_mulhi.restype = C.c_uint32
        L.orc_mulhi.argtypes = [C.c_uint32, C.c_uint32]
        L.orc_init_chain.argtypes = [C.c_void_p, C.c_uint64, C.c_uint32, C.c_void_p]
        L.orc_propose.argtypes = [C.c_uint32, C.c_uint32, C.c_int, C.c_int, C.c_int, C.c_void_p,
                                  C.c_void_p, C.c_void_p]
        L.orc_accept.restype = C.c_int
        L.orc_accept.argtypes = [C.c_int64, C.c_uint32, C.c_void_p, C.c_int]
        L.orc_run_chain.argtypes = [C.c_void_p, C.c_uint64, C.c_uint32, C.c_uint64, C.c_int64, C.c_int,
                                    C.c_int64, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p,
                                    C.c_void_p, C.c_void_p]
        L.orc_geometric_table.argtypes = [C.c_double, C.c_double, C.c_int, C.c_int, C.c_void_p]
        L.orc_valid.restype = C.c_int
        L.orc_valid.argtypes = [C.c_void_p, C.c_void_p]
        L.orc_init_chain_c.argtypes = [C.c_void_p, C.c_uint64, C.c_uint32, C.c_void_p]
        L.orc_propose_c.restype = C.c_int
        L.orc_propose_c.argtypes = [C.c_void_p, C.c_uint32, C.c_uint32, C.c_void_p, C.c_void_p, C.c_void_p]
        L.orc_run_chain_c.argtypes = L.orc_run_chain.argtypes
        _lib = L
    return _lib


def philox4x32_10(ctr: Sequence[int], key: Sequence[int]) -> List[int]:
    c = np.array(ctr, dtype=np.uint32)
    k = np.array(key, dtype=np.uint32)
    o = np.zeros(4, dtype=np.uint32)
    lib().orc_philox4x32_10(c.ctypes.data, k.ctypes.data, o.ctypes.data)
    return [int(v) for v in o]


def mulhi(a: int, b: int) -> int:
    return int(lib().orc_mulhi(a, b))


def propose(x0: int, x1: int, n_params: int, n_edges: int, n_pairs: int, cur: np.ndarray):
    cur = np.ascontiguousarray(cur, dtype=np.int8)
    p, nv = C.c_int32(), C.c_int32()
    lib().orc_propose(x0, x1, n_params, n_edges, n_pairs, cur.ctypes.data, C.byref(p), C.byref(nv))
    return p.value, nv.value


def accept(d: int, x2: int, row: np.ndarray) -> bool:
    row = np.ascontiguousarray(row, dtype=np.uint32)
    return bool(lib().orc_accept(d, x2, row.ctypes.data, row.shape[0]))


def geometric_table(t0: float, t_end: float, n_levels: int, dmax: int) -> np.ndarray:
    out = np.zeros((n_levels, dmax), dtype=np.uint32)
    lib().orc_geometric_table(t0, t_end, n_levels, dmax, out.ctypes.data)
    return out


def unpack_trace(rec: np.ndarray):
    """u64 trace records -> dict of arrays (delta_cand, param, code, accepted, new_best)."""
    rec = np.asarray(rec, dtype=np.uint64)
    return {
        "delta_cand": (rec & np.uint64(0xFFFFFFFF)).astype(np.uint32),
        "param": ((rec >> np.uint64(32)) & np.uint64(0xFFFFFF)).astype(np.int64),
        "code": ((rec >> np.uint64(56)) & np.uint64(0xF)).astype(np.int64),
        "accepted": ((rec >> np.uint64(60)) & np.uint64(1)).astype(bool),
        "new_best": ((rec >> np.uint64(61)) & np.uint64(1)).astype(bool),
        "null_move": ((rec >> np.uint64(62)) & np.uint64(1)).astype(bool),
    }


class Oracle:
    """The oracle bound to one problem (any object with the fields of problems.Problem)."""

    def __init__(self, prob):
        self.prob = prob
        self._keep = [np.ascontiguousarray(prob.edge_src, dtype=np.int32),
                      np.ascontiguousarray(prob.edge_dst, dtype=np.int32),
                      np.ascontiguousarray(prob.th_lo, dtype=np.int8),
                      np.ascontiguousarray(prob.th_hi, dtype=np.int8),
                      np.ascontiguousarray(prob.obs_times, dtype=np.int32),
                      np.ascontiguousarray(prob.init_state, dtype=np.uint8),
                      np.ascontiguousarray(prob.clamp, dtype=np.uint8),
                      np.ascontiguousarray(prob.obs, dtype=np.uint8)]
        s, d, lo, hi, ot, ini, cl, ob = self._keep
        self.N, self.E, self.K, self.T = prob.n_nodes, prob.n_edges, prob.n_cond, prob.n_steps
        self.n_obs = int(ot.shape[0])
        self.P = self.E + self.N
        self.h = lib().orc_problem_create(self.N, self.E, s.ctypes.data, d.ctypes.data, int(lo.shape[0]),
                                          lo.ctypes.data, hi.ctypes.data, self.K, self.T, self.n_obs,
                                          ot.ctypes.data, ini.ctypes.data, cl.ctypes.data, ob.ctypes.data)

    def __del__(self):
        try:
            if self.h:
                lib().orc_problem_destroy(self.h)
                self.h = None
        except Exception:
            pass

    def _params(self, x) -> np.ndarray:
        x = np.ascontiguousarray(x, dtype=np.int8)
        assert x.shape[-1] == self.P, "parameter vector has the wrong length"
        return x

    def fitness(self, params) -> int:
        x = self._params(params)
        return int(lib().orc_fitness(self.h, x.ctypes.data))

    def simulate(self, params) -> np.ndarray:
        """Full trajectory uint8 [K][T+1][N] (t = 0 is the initial state)."""
        x = self._params(params)
        traj = np.zeros((self.K, self.T + 1, self.N), dtype=np.uint8)
        lib().orc_simulate(self.h, x.ctypes.data, traj.ctypes.data)
        return traj

    def states_at_obs(self, params) -> np.ndarray:
        """uint8 [K][n_obs][N]: the simulated states at the observation times."""
        traj = self.simulate(params)
        return np.ascontiguousarray(traj[:, np.asarray(self.prob.obs_times, dtype=np.int64), :])

    def fitness_batch(self, params, threads: int = 1) -> np.ndarray:
        x = self._params(params).reshape(-1, self.P)
        out = np.zeros(x.shape[0], dtype=np.uint32)
        if threads <= 1 or x.shape[0] < 2 * threads:
            lib().orc_fitness_batch(self.h, x.ctypes.data, x.shape[0], out.ctypes.data)
            return out
        # the same single-threaded code replicated over independent parameter sets
        bounds = np.linspace(0, x.shape[0], threads + 1).astype(np.int64)

        def work(t):
            a, b = int(bounds[t]), int(bounds[t + 1])
            if b > a:
                lib().orc_fitness_batch(self.h, x[a:b].ctypes.data, b - a, out[a:b].ctypes.data)
        with ThreadPoolExecutor(threads) as ex:
            list(ex.map(work, range(threads)))
        return out

    def init_chain(self, seed: int, chain: int, constrained: bool = False):
        x = np.zeros(self.P, dtype=np.int8)
        if constrained:
            indeg = np.bincount(self._keep[1], minlength=self.N)
            outdeg = np.bincount(self._keep[0], minlength=self.N)
            if (indeg == 0).any() or (outdeg == 0).any():       # no valid vector exists
                raise ValueError("constraints need an in-edge and an out-edge at every node")
            lib().orc_init_chain_c(self.h, seed, chain, x.ctypes.data)
        else:
            lib().orc_init_chain(self.h, seed, chain, x.ctypes.data)
        return x, self.fitness(x)

    def valid(self, params) -> bool:
        """Structural constraints (a) and (b) of PAPER.md:186-199 in this model (reading C1)."""
        return bool(lib().orc_valid(self.h, self._params(params).ctypes.data))

    def propose_c(self, x0: int, x1: int, cur):
        """Constrained GetCandidate -> (parameter index, new value, moved)."""
        cur = self._params(cur)
        p, nv = C.c_int32(), C.c_int32()
        moved = lib().orc_propose_c(self.h, x0, x1, cur.ctypes.data, C.byref(p), C.byref(nv))
        return p.value, nv.value, bool(moved)

    def run_chain(self, sched, chain: int, n_steps: int, g0: int = 0, state=None, trace: bool = True,
                  constrained: bool = False):
        """Advance global chain id ``chain`` by n_steps from step g0.

        state = (cur, best, fit_cur, fit_best) or None (= fresh chain).
        Returns dict(cur, best, fit_cur, fit_best, trace, init_fit).
        """
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
        run = lib().orc_run_chain_c if constrained else lib().orc_run_chain
        run(self.h, sched.seed, chain, g0, n_steps, sched.n_levels, sched.steps_per_level,
            sched.dmax, table.ctypes.data, cur.ctypes.data, best.ctypes.data,
            C.byref(fcur), C.byref(fbest), tr.ctypes.data if trace else None)
        return {"cur": cur, "best": best, "fit_cur": fcur.value, "fit_best": fbest.value,
                "trace": tr, "init_fit": f0}

    def run_chains(self, sched, chains: Iterable[int], n_steps: int, threads: int = 1, trace: bool = True,
                   constrained: bool = False):
        """Independent chains, optionally replicated over host threads (ctypes drops the GIL)."""
        chains = list(chains)
        if threads <= 1:
            return [self.run_chain(sched, c, n_steps, trace=trace, constrained=constrained) for c in chains]
        with ThreadPoolExecutor(threads) as ex:
            return list(ex.map(lambda c: self.run_chain(sched, c, n_steps, trace=trace, constrained=constrained), chains))


def run_levels(orc: "Oracle", sched, n_chains: int, n_levels: int, group_size: int = 0, g0: int = 0,
               states=None, threads: int = 1, constrained: bool = False):
    """PAPER.md Table 1 (:125-155), the level structure around the chain step, statement by statement:

        while T > T_min:                                   # here: n_levels levels from step g0
            for every thread: n_iterations chain steps     # steps_per_level x Oracle.run_chain (c-3)
            d*_best = min_i d_best(i)                      # :150-151, per group; ties -> smallest chain
            every x_best(i) = x*_best                      # :152-153
            T = rho T                                      # level index from the step counter (reading 6)
        (top of the next level: d_current = d_best; x_current = x_best, :129)

    group_size = 0: one group of all chains (the paper); else groups of consecutive chains (its
    future work, :321).  states = list of (cur, best, fit_cur, fit_best) per chain or None (fresh
    chains, global ids chain_id_base + i).  Returns the list of states after the last level.
    """
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
            star = min(members, key=lambda c: (states[c][3], c))          # smallest d_best, then smallest chain
            x_star, d_star = states[star][1], states[star][3]
            for c in members:
                states[c] = (x_star.copy(), x_star.copy(), d_star, d_star)
    return states


def simulate_fn(prob, params) -> np.ndarray:
    """The ``simulate`` callback problems.make_problem expects, served by the oracle."""
    return Oracle(prob).states_at_obs(params)
