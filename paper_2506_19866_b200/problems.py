"""Seeded synthetic inputs for the ternary-logic SA hot path.

This module is the ONE piece shared by the CUDA path, the CPU oracle, the tests
and bench.py.  It holds none of the method's arithmetic: it never updates a
network state, never scores a trajectory and never draws an SA random number.
Where the recipe needs a simulated time course (the hidden ground truth is
simulated to make the observations, "we use the Simulate()
function of our code to generate a pseudo-experimental time series") the caller
injects a ``simulate`` callback: tests pass the oracle's, bench.py passes the
CUDA library's ``sa_simulate``.

Recipe: SURVEY.md §8(d) "Synthetic inputs" / DESIGN.md §4.  The five configs are
BASELINE.json's ``configs``.  The paper's own HPG / Mtb edge lists and data
 are not available; these stand in for them, taking their
shape (parameter counts 102 and ~10x that, ~5/9 of the nodes observed,
self-generated reference data from hidden parameters).
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field
from typing import Callable, Dict, List, Optional

import numpy as np

MASK64 = (1 << 64) - 1
UNOBSERVED = 255

# reading 5: the six (t_lo, t_hi) pairs, t_lo < t_hi, in [-3, 3]
TH_LO = (-3, -2, -1, 0, 0, 1)
TH_HI = (-1, 0, 0, 1, 2, 3)


class SplitMix64:
    """Tiny counter-style generator used only to make inputs (never by the method)."""

    def __init__(self, seed: int, stream: int = 0):
        self.state = (seed * 0x9E3779B97F4A7C15 + (stream + 1) * 0xD1B54A32D192ED03) & MASK64

    def next(self) -> int:
        self.state = (self.state + 0x9E3779B97F4A7C15) & MASK64
        z = self.state
        z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & MASK64
        z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & MASK64
        return z ^ (z >> 31)

    def below(self, n: int) -> int:
        """Uniform integer in [0, n) (integer-only; bias < 2^-32)."""
        return ((self.next() >> 32) * n) >> 32

    def uniform(self) -> float:
        return (self.next() >> 11) * (1.0 / (1 << 53))

    def sample_distinct(self, n: int, k: int) -> List[int]:
        """k distinct integers from [0, n), order of draw kept."""
        if k > n:
            raise ValueError("sample larger than population")
        if 3 * k < n:  # rejection
            seen, out = set(), []
            while len(out) < k:
                v = self.below(n)
                if v not in seen:
                    seen.add(v)
                    out.append(v)
            return out
        pool = list(range(n))  # partial Fisher-Yates
        for i in range(k):
            j = i + self.below(n - i)
            pool[i], pool[j] = pool[j], pool[i]
        return pool[:k]


@dataclass(frozen=True)
class ConfigSpec:
    name: str
    seed: int
    n_nodes: int
    n_edges: int
    degree: str          # "uniform-pairs" | "poisson" | "powerlaw"
    n_cond: int
    n_clamped: int
    n_steps: int
    obs_times: tuple
    n_chains: int
    sa_steps: int
    max_in_degree: int = 0   # 0 = N-1


def _times(first, last, step):
    return tuple(range(first, last + 1, step))


# BASELINE.json configs 1..5 (config 4 = "scaling" reuses the Mtb-shaped problem)
CONFIGS: Dict[str, ConfigSpec] = {
    "tiny": ConfigSpec("tiny", 1001, 8, 20, "uniform-pairs", 2, 1, 12, _times(3, 12, 3), 8, 2000),
    "hpg": ConfigSpec("hpg", 1002, 18, 84, "poisson", 4, 2, 24, _times(3, 24, 3), 1024, 20000),
    "mtb": ConfigSpec("mtb", 1003, 100, 900, "powerlaw", 8, 3, 32, _times(4, 32, 4), 4096, 20000, 40),
    "large": ConfigSpec("large", 1005, 1000, 10000, "poisson", 16, 5, 32, _times(4, 32, 4), 2048, 1000),
}
SCALING_CHAINS = (1024, 8192, 65536)   # config 4, on "mtb"
SCALING_STEPS = 2000
SA_SEED = 42
T0, T_END, N_LEVELS, DMAX = 4.0, 0.05, 200, 64


@dataclass
class Problem:
    name: str
    seed: int
    n_nodes: int
    n_edges: int
    edge_src: np.ndarray      # int32 [E] caller's edge order
    edge_dst: np.ndarray      # int32 [E]
    th_lo: np.ndarray         # int8 [n_pairs]
    th_hi: np.ndarray         # int8 [n_pairs]
    n_cond: int
    n_steps: int
    obs_times: np.ndarray     # int32 [n_obs], strictly increasing, in [1, T]
    init_state: np.ndarray    # uint8 [K][N] in {0,1,2}
    clamp: np.ndarray         # uint8 [K][N] 0/1
    obs: np.ndarray           # uint8 [K][n_obs][N] in {0,1,2} or 255 (= unobserved)
    truth: Optional[np.ndarray] = None         # int8 [E+N] hidden ground truth
    obs_clean: Optional[np.ndarray] = None     # obs before the flips
    observed_nodes: Optional[np.ndarray] = None
    n_flipped: int = 0
    meta: dict = field(default_factory=dict)

    @property
    def n_pairs(self) -> int:
        return int(self.th_lo.shape[0])

    @property
    def n_obs(self) -> int:
        return int(self.obs_times.shape[0])

    @property
    def n_params(self) -> int:
        return self.n_edges + self.n_nodes

    @property
    def node_updates_per_step(self) -> int:
        """Nominal K*T*N of SURVEY.md §8 (clamped nodes included)."""
        return self.n_cond * self.n_steps * self.n_nodes

    @property
    def n_scored(self) -> int:
        return int((self.obs != UNOBSERVED).sum())

    @property
    def alg_ops_per_step(self) -> int:
        """A_alg = K*T*(E+3N) + K*n_obs*N_obs."""
        return self.n_cond * self.n_steps * (self.n_edges + 3 * self.n_nodes) + self.n_scored


@dataclass
class Schedule:
    n_chains: int
    seed: int
    n_levels: int
    steps_per_level: int
    dmax: int
    accept: np.ndarray        # uint32 [L][D]
    total_steps: int
    chain_id_base: int = 0    # global id of local chain 0 (multi-GPU chain-range partition)


def geometric_table(t0: float, t_end: float, n_levels: int, dmax: int) -> np.ndarray:
    """Acceptance thresholds floor(2^32 * exp(-d / T_l)), d = 1..dmax (input data).

    T_l = t0 * (t_end/t0)^(l/(L-1)); T_0 = t0 when L == 1.  Clamped to 2^32-1.
    """
    out = np.zeros((n_levels, dmax), dtype=np.uint32)
    for l in range(n_levels):
        temp = t0 if n_levels == 1 else t0 * math.pow(t_end / t0, l / (n_levels - 1))
        for d in range(1, dmax + 1):
            v = math.floor(4294967296.0 * math.exp(-d / temp))
            out[l, d - 1] = min(v, 0xFFFFFFFF)
    return out


def make_schedule(n_chains: int, total_steps: int, seed: int = SA_SEED,
                  t0: float = T0, t_end: float = T_END, n_levels: int = N_LEVELS,
                  dmax: int = DMAX, chain_id_base: int = 0) -> Schedule:
    spl = max(1, total_steps // n_levels)
    return Schedule(n_chains, seed, n_levels, spl, dmax,
                    geometric_table(t0, t_end, n_levels, dmax), total_steps, chain_id_base)


def default_schedule(name: str, n_chains: Optional[int] = None,
                     total_steps: Optional[int] = None) -> Schedule:
    spec = CONFIGS[name]
    return make_schedule(n_chains or spec.n_chains, total_steps or spec.sa_steps)


# --------------------------------------------------------------------------- structure

def _poisson(rng: SplitMix64, lam: float) -> int:
    u = rng.uniform()
    k, p = 0, math.exp(-lam)
    cdf = p
    while u > cdf and k < 10000:
        k += 1
        p *= lam / k
        cdf += p
    return k


def _powerlaw_table(lo: int, hi: int, gamma: float):
    w = [k ** (-gamma) for k in range(lo, hi + 1)]
    tot = sum(w)
    cdf, acc = [], 0.0
    for x in w:
        acc += x / tot
        cdf.append(acc)
    return cdf


def _draw_degrees(spec: ConfigSpec, rng: SplitMix64) -> List[int]:
    n, e = spec.n_nodes, spec.n_edges
    dmax = min(n - 1, spec.max_in_degree or (n - 1))
    if spec.degree == "poisson":
        deg = [_poisson(rng, e / n) for _ in range(n)]
    else:  # P(k) ~ k^-2.2 on [4, 40] (reading 22)
        cdf = _powerlaw_table(4, 40, 2.2)
        deg = []
        for _ in range(n):
            u = rng.uniform()
            k = 0
            while k < len(cdf) - 1 and u > cdf[k]:
                k += 1
            deg.append(4 + k)
    deg = [min(max(d, 1), dmax) for d in deg]
    total = sum(deg)
    while total != e:  # +-1 on random nodes within bounds until the sum is E
        i = rng.below(n)
        if total < e and deg[i] < dmax:
            deg[i] += 1
            total += 1
        elif total > e and deg[i] > 1:
            deg[i] -= 1
            total -= 1
    return deg


def _make_edges(spec: ConfigSpec, rng: SplitMix64):
    n, e = spec.n_nodes, spec.n_edges
    pairs = []
    if spec.degree == "uniform-pairs":
        # E distinct ordered pairs (src != dst), uniform without replacement; in-degree 0 may occur
        for code in rng.sample_distinct(n * (n - 1), e):
            s, r = divmod(code, n - 1)
            d = r if r < s else r + 1
            pairs.append((s, d))
    else:
        deg = _draw_degrees(spec, rng)
        for i in range(n):
            for v in rng.sample_distinct(n - 1, deg[i]):
                pairs.append((v if v < i else v + 1, i))
        # repair out-degree 0: re-point the source of an edge whose source has out-degree >= 2
        outdeg = [0] * n
        have = set(pairs)
        for s, _ in pairs:
            outdeg[s] += 1
        for v in range(n):
            tries = 0
            while outdeg[v] == 0 and tries < 100000:
                tries += 1
                k = rng.below(len(pairs))
                s, d = pairs[k]
                if outdeg[s] >= 2 and d != v and (v, d) not in have:
                    have.discard((s, d))
                    have.add((v, d))
                    pairs[k] = (v, d)
                    outdeg[s] -= 1
                    outdeg[v] += 1
        # caller's edge order is a random permutation (not grouped by destination)
        order = rng.sample_distinct(len(pairs), len(pairs))
        pairs = [pairs[k] for k in order]
    src = np.array([p[0] for p in pairs], dtype=np.int32)
    dst = np.array([p[1] for p in pairs], dtype=np.int32)
    return src, dst


SimulateFn = Callable[[Problem, np.ndarray], np.ndarray]
"""simulate(problem, params int8[E+N]) -> uint8 [K][n_obs][N]: states at the observation times."""


def make_problem(name: str, simulate: SimulateFn, seed: Optional[int] = None,
                 noise: float = 0.05, spec: Optional[ConfigSpec] = None) -> Problem:
    """Build one of the five configs deterministically from (name, seed).

    ``simulate`` supplies the states of a parameter set at the observation times; it is
    the only place the method's arithmetic enters and it is never defined here.
    """
    spec = spec or CONFIGS[name]
    seed = spec.seed if seed is None else seed
    n, e, kc, nobs = spec.n_nodes, spec.n_edges, spec.n_cond, len(spec.obs_times)

    src, dst = _make_edges(spec, SplitMix64(seed, 1))

    # conditions: random initial state, c distinct clamped nodes whose value is drawn from {0, 2}
    rng = SplitMix64(seed, 2)
    init = np.zeros((kc, n), dtype=np.uint8)
    clamp = np.zeros((kc, n), dtype=np.uint8)
    for k in range(kc):
        for i in range(n):
            init[k, i] = rng.below(3)
        for i in rng.sample_distinct(n, spec.n_clamped):
            clamp[k, i] = 1
            init[k, i] = 2 * rng.below(2)

    # observed node subset: round(5N/9), same in every condition and time (reading 10)
    rng = SplitMix64(seed, 3)
    n_observed = int(round(5 * n / 9))
    observed = np.array(sorted(rng.sample_distinct(n, n_observed)), dtype=np.int32)

    prob = Problem(name=spec.name, seed=seed, n_nodes=n, n_edges=e, edge_src=src, edge_dst=dst,
                   th_lo=np.array(TH_LO, dtype=np.int8), th_hi=np.array(TH_HI, dtype=np.int8),
                   n_cond=kc, n_steps=spec.n_steps,
                   obs_times=np.array(spec.obs_times, dtype=np.int32),
                   init_state=init, clamp=clamp,
                   obs=np.full((kc, nobs, n), UNOBSERVED, dtype=np.uint8),
                   observed_nodes=observed)

    # hidden ground truth: resample (<= 100 tries) until >= 30 % of observed node time courses
    # are non-constant in some condition (the paper preferred dynamic nodes)
    rng = SplitMix64(seed, 4)
    best_frac, truth, states = -1.0, None, None
    for attempt in range(100):
        cand = np.zeros(e + n, dtype=np.int8)
        for p in range(e):
            cand[p] = rng.below(3) - 1
        for i in range(n):
            cand[e + i] = rng.below(len(TH_LO))
        st = np.asarray(simulate(prob, cand), dtype=np.uint8).reshape(kc, nobs, n)
        sub = st[:, :, observed]                                 # [K][n_obs][N_obs]
        dynamic = (sub.max(axis=1) != sub.min(axis=1)).any(axis=0)
        frac = float(dynamic.mean())
        if frac > best_frac:
            best_frac, truth, states = frac, cand, st
        if frac >= 0.30:
            break
    prob.truth = truth
    prob.meta["dynamic_fraction"] = best_frac
    prob.meta["truth_attempts"] = attempt + 1

    clean = np.full((kc, nobs, n), UNOBSERVED, dtype=np.uint8)
    clean[:, :, observed] = states[:, :, observed]
    prob.obs_clean = clean

    # noise: exactly round(noise * #observed entries) entries, without replacement, each set to
    # one of the two other levels with equal probability (reading 13)
    rng = SplitMix64(seed, 5)
    noisy = clean.copy()
    n_entries = kc * nobs * n_observed
    n_flip = int(round(noise * n_entries))
    for code in rng.sample_distinct(n_entries, n_flip):
        k, rem = divmod(code, nobs * n_observed)
        j, oi = divmod(rem, n_observed)
        i = int(observed[oi])
        noisy[k, j, i] = (int(noisy[k, j, i]) + 1 + rng.below(2)) % 3
    prob.obs = noisy
    prob.n_flipped = n_flip
    return prob


def random_params(prob: Problem, count: int, seed: int) -> np.ndarray:
    """count i.i.d. uniform parameter vectors int8 [count][E+N] (inputs for sa_eval parity)."""
    rng = np.random.Generator(np.random.Philox(seed))
    w = rng.integers(-1, 2, size=(count, prob.n_edges), dtype=np.int8)
    th = rng.integers(0, prob.n_pairs, size=(count, prob.n_nodes), dtype=np.int8)
    return np.ascontiguousarray(np.concatenate([w, th], axis=1))


def spread_chains(n_chains: int, count: int, head: int = 4) -> List[int]:
    """Parity subsets of SURVEY §8(d): the first ``head`` chains plus evenly spread ones."""
    ids = list(range(min(head, n_chains)))
    rest = count - len(ids)
    for k in range(rest):
        ids.append(min(n_chains - 1, head + ((n_chains - head) * k) // max(rest, 1)))
    return sorted(set(ids))


# =========================================================================== paper model
# Inputs for the paper's OWN model (§2.1-2.3, §2.5): three
# parameters per edge (w, p, t), three per node (u, m, d), one time course of T+1 points per
# condition, a reference matrix R with 255 = entity not measured.  As above, nothing here updates a
# state or scores a trajectory: the ground-truth time course comes from the injected callback.

@dataclass(frozen=True)
class PaperSpec:
    name: str
    seed: int
    n_nodes: int
    n_edges: int
    n_measured: int
    n_fast: int
    n_cond: int
    n_steps: int             # T transitions = T+1 time points including t0
    noise: float
    n_chains: int
    sa_steps: int


# The paper's two systems by SHAPE (their edge lists and data are not in the container): HPG axis
# 9 nodes / 25 edges / 102 parameters, 5 of 9 measured, FSH / GNRH1 / LH fast, 20 time points,
# experimental (hence imperfectly fitting) data; Mtb 63 / 178 / 723, 35
# measured, one third fast, 20 time points, self-generated noise-free data (:182-184).
PAPER_CONFIGS: Dict[str, PaperSpec] = {
    "paper_tiny": PaperSpec("paper_tiny", 2001, 5, 11, 3, 2, 2, 9, 0.05, 8, 2000),
    "paper_hpg": PaperSpec("paper_hpg", 2002, 9, 25, 5, 3, 1, 19, 0.05, 10240, 5000),
    "paper_mtb": PaperSpec("paper_mtb", 2003, 63, 178, 35, 21, 1, 19, 0.0, 10240, 5000),
}
PAPER_T0, PAPER_TMIN, PAPER_RHO, PAPER_ITERS = 1000.0, 0.001, 0.99, 5000


@dataclass
class PaperProblem:
    name: str
    seed: int
    n_nodes: int
    n_edges: int
    edge_src: np.ndarray      # int32 [E]
    edge_dst: np.ndarray      # int32 [E]
    fast: np.ndarray          # uint8 [N] 1 = speed range {10,11,12}, 0 = {1..6}
    n_cond: int
    n_steps: int              # T
    init_state: np.ndarray    # uint8 [K][N]
    ref: np.ndarray           # uint8 [K][T+1][N] in {0,1,2} or 255
    truth: Optional[np.ndarray] = None
    ref_clean: Optional[np.ndarray] = None
    measured_nodes: Optional[np.ndarray] = None
    n_flipped: int = 0
    meta: dict = field(default_factory=dict)

    @property
    def n_params(self) -> int:
        return 3 * self.n_edges + 3 * self.n_nodes

    @property
    def n_scored(self) -> int:
        return int((self.ref != UNOBSERVED).sum())

    @property
    def max_objective(self) -> int:
        """Upper bound of y: |S-R| <= 2 and |G|+1 <= 3 per measured entry."""
        return 6 * self.n_scored

    @property
    def node_updates_per_step(self) -> int:
        return self.n_cond * self.n_steps * self.n_nodes

    @property
    def alg_ops_per_step(self) -> int:
        """Scalar integer operations one chain-step must do: per transition one
        multiply-add per edge (image) and 8 per node (clip, compare, memory test, priority product,
        maximum, equality with the maximum, bounded move, counter update), plus one
        absolute-difference-multiply-add per measured entry of every time point."""
        return self.n_cond * self.n_steps * (self.n_edges + 8 * self.n_nodes) + self.n_scored

    def layout(self):
        """Offsets of w, p, t, u, m, d in the parameter vector."""
        e, n = self.n_edges, self.n_nodes
        return {"w": 0, "p": e, "t": 2 * e, "u": 3 * e, "m": 3 * e + n, "d": 3 * e + 2 * n}


def paper_domain(prob: PaperProblem, q: int):
    """Values parameter q may take, in increasing order."""
    e, n = prob.n_edges, prob.n_nodes
    if q < e:
        return (0, 1, 2)
    if q < 2 * e:
        return (-1, 0, 1)
    if q < 3 * e:
        return (1, 2)
    q -= 3 * e
    if q < n:
        return (10, 11, 12) if prob.fast[q] else (1, 2, 3, 4, 5, 6)
    if q < 2 * n:
        return (0, 1, 2)
    return (1, 2)


def paper_schedule(n_chains: int, n_levels: int, steps_per_level: int, dmax: int, seed: int = SA_SEED,
                   t0: float = PAPER_T0, rho: float = PAPER_RHO, chain_id_base: int = 0) -> Schedule:
    """The paper's cooling T_l = t0 * rho^l as an integer acceptance table
    floor(2^32 * exp(-d / T_l)), d = 1..dmax.  The full schedule is 1375 levels x 5000 iterations
    (T = 1000 down to 0.001); tests and bench.py run slices of it."""
    out = np.zeros((n_levels, dmax), dtype=np.uint32)
    d = np.arange(1, dmax + 1, dtype=np.float64)
    for l in range(n_levels):
        temp = t0 * math.pow(rho, l)
        v = np.floor(4294967296.0 * np.exp(-d / temp))
        out[l] = np.minimum(v, 4294967295.0).astype(np.uint32)
    return Schedule(n_chains, seed, n_levels, steps_per_level, dmax, out, n_levels * steps_per_level, chain_id_base)


def paper_levels(t0: float = PAPER_T0, tmin: float = PAPER_TMIN, rho: float = PAPER_RHO) -> int:
    """Number of passes of `while T > Tmin`: 1375 for the paper's constants."""
    n, t = 0, t0
    while t > tmin:
        n += 1
        t *= rho
    return n


PaperSimulateFn = Callable[[PaperProblem, np.ndarray], np.ndarray]
"""simulate(problem, params int8[3E+3N]) -> uint8 [K][T+1][N]: the whole time course, t0 included."""


def make_paper_problem(name: str, simulate: PaperSimulateFn, seed: Optional[int] = None,
                       spec: Optional[PaperSpec] = None) -> PaperProblem:
    spec = spec or PAPER_CONFIGS[name]
    seed = spec.seed if seed is None else seed
    n, e, kc, T = spec.n_nodes, spec.n_edges, spec.n_cond, spec.n_steps

    # candidate structure: every node has an in- and an out-edge (closed loop)
    shape = ConfigSpec(spec.name, seed, n, e, "poisson", kc, 0, T, (), 0, 0)
    src, dst = _make_edges(shape, SplitMix64(seed, 1))

    rng = SplitMix64(seed, 2)
    init = np.zeros((kc, n), dtype=np.uint8)
    for k in range(kc):
        for i in range(n):
            init[k, i] = rng.below(3)
    fast = np.zeros(n, dtype=np.uint8)
    for i in SplitMix64(seed, 3).sample_distinct(n, spec.n_fast):
        fast[i] = 1

    prob = PaperProblem(name=spec.name, seed=seed, n_nodes=n, n_edges=e, edge_src=src, edge_dst=dst, fast=fast,
                        n_cond=kc, n_steps=T, init_state=init,
                        ref=np.full((kc, T + 1, n), UNOBSERVED, dtype=np.uint8))

    # hidden ground truth: uniform over the value ranges, made constraint-compliant by giving every
    # node one activating in-edge and one non-zero out-edge ("randomized within their
    # specified ranges ... adhere to the network constraints"); resampled (<= 100 tries) until
    # >= 30 % of the nodes have a non-constant time course
    rng = SplitMix64(seed, 4)
    in_edges = [[k for k in range(e) if dst[k] == i] for i in range(n)]
    out_edges = [[k for k in range(e) if src[k] == i] for i in range(n)]
    best_frac, truth, states = -1.0, None, None
    for attempt in range(100):
        cand = np.zeros(3 * e + 3 * n, dtype=np.int8)
        for q in range(3 * e + 3 * n):
            dom = paper_domain(prob, q)
            cand[q] = dom[rng.below(len(dom))]
        for i in range(n):
            k = in_edges[i][rng.below(len(in_edges[i]))]
            cand[e + k] = 1
            cand[k] = max(int(cand[k]), 1)
        for i in range(n):
            if not any(cand[k] > 0 for k in out_edges[i]):
                cand[out_edges[i][rng.below(len(out_edges[i]))]] = 1
        st = np.asarray(simulate(prob, cand), dtype=np.uint8).reshape(kc, T + 1, n)
        dynamic = (st.max(axis=1) != st.min(axis=1)).any(axis=0)
        frac = float(dynamic.mean())
        if frac > best_frac:
            best_frac, truth, states = frac, cand, st
        if frac >= 0.30:
            break
    prob.truth = truth
    prob.meta["dynamic_fraction"] = best_frac
    prob.meta["truth_attempts"] = attempt + 1

    # measured subset: dynamic nodes first, then the others, each group in random order (:184 "mostly
    # randomly selected; however, we prioritize ... a more dynamic time course")
    rng = SplitMix64(seed, 5)
    dynamic = (states.max(axis=1) != states.min(axis=1)).any(axis=0)
    order = rng.sample_distinct(n, n)
    ranked = [i for i in order if dynamic[i]] + [i for i in order if not dynamic[i]]
    measured = np.array(sorted(ranked[:spec.n_measured]), dtype=np.int32)
    prob.measured_nodes = measured
    clean = np.full((kc, T + 1, n), UNOBSERVED, dtype=np.uint8)
    clean[:, :, measured] = states[:, :, measured]
    prob.ref_clean = clean

    rng = SplitMix64(seed, 6)
    noisy = clean.copy()
    n_entries = kc * (T + 1) * len(measured)
    n_flip = int(round(spec.noise * n_entries))
    for code in rng.sample_distinct(n_entries, n_flip):
        k, rem = divmod(code, (T + 1) * len(measured))
        t, oi = divmod(rem, len(measured))
        i = int(measured[oi])
        noisy[k, t, i] = (int(noisy[k, t, i]) + 1 + rng.below(2)) % 3
    prob.ref = noisy
    prob.n_flipped = n_flip
    return prob


def random_paper_params(prob: PaperProblem, count: int, seed: int) -> np.ndarray:
    """count i.i.d. uniform parameter vectors int8 [count][3E+3N] (inputs for sap_eval parity)."""
    rng = np.random.Generator(np.random.Philox(seed))
    out = np.zeros((count, prob.n_params), dtype=np.int8)
    for q in range(prob.n_params):
        dom = np.array(paper_domain(prob, q), dtype=np.int8)
        out[:, q] = dom[rng.integers(0, len(dom), size=count)]
    return out
