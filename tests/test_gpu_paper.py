"""Parity of the paper-model CUDA path (sap_* through the C ABI) against the paper-model CPU oracle —
bit-exact, element by element, on the same seeded inputs.
Everything here needs a GPU (-m gpu)."""
import copy
import os
from concurrent.futures import ThreadPoolExecutor

import numpy as np
import pytest

from oracle import oracle_paper as OP
from paper_2506_19866_b200 import problems as PB
from paper_2506_19866_b200.telemetry import acceptance_by_level
from helpers import golden_rows
from test_oracle_paper_pins import example_c

pytestmark = pytest.mark.gpu
NCPU = max(1, min(32, os.cpu_count() or 1))


@pytest.fixture(scope="module")
def B():
    import torch
    assert torch.cuda.is_available(), "the gpu tests need a CUDA device"
    from paper_2506_19866_b200 import build
    build.build()
    from paper_2506_19866_b200 import binding
    binding.use_torch_plumbing()
    return binding


@pytest.fixture(scope="module")
def paper_problems():
    cache = {}

    def get(name):
        if name not in cache:
            cache[name] = PB.make_paper_problem(name, OP.simulate_fn)
        return cache[name]
    return get


class Handle:
    def __init__(self, B, prob, sched, flags=0):
        self.B, self.prob, self.sched, self.flags = B, prob, sched, flags
        self.h = B.sap_create(prob, sched, flags)

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.B.sap_destroy(self.h)


def oracle_chains(orc, sched, chains, n_steps, constrained):
    with ThreadPoolExecutor(NCPU) as ex:
        return list(ex.map(lambda c: orc.run_chain(sched, c + sched.chain_id_base, n_steps, constrained=constrained), chains))


def check_chains(B, hd, orc, chains, n_steps, trace=None):
    con = bool(hd.flags & B.SAP_CONSTRAINED)
    refs = oracle_chains(orc, hd.sched, chains, n_steps, con)
    for row, (c, ref) in enumerate(zip(chains, refs)):
        cur, fc, best, fb = B.sap_get_chain(hd.h, c, hd.prob.n_params)
        if trace is not None:
            bad = np.nonzero(trace[row][:n_steps] != ref["trace"])[0]
            assert bad.size == 0, f"chain {c}: first trace mismatch at step {bad[0]}: " \
                                  f"gpu {int(trace[row][bad[0]]):#x} oracle {int(ref['trace'][bad[0]]):#x}"
        assert (fc, fb) == (ref["fit_cur"], ref["fit_best"]), f"chain {c} fitness"
        assert np.array_equal(cur, ref["cur"]), f"chain {c} current vector"
        assert np.array_equal(best, ref["best"]), f"chain {c} best vector"
        if con:
            assert orc.valid(cur) and orc.valid(best)


def check_all_fitness(B, hd, orc):
    R, P = hd.sched.n_chains, hd.prob.n_params
    fcur, fbest = B.sap_get_fitness(hd.h, R)
    assert (fbest <= fcur).all()
    cur = np.zeros((R, P), dtype=np.int8)
    best = np.zeros((R, P), dtype=np.int8)
    for c in range(R):
        cur[c], fc, best[c], fb = B.sap_get_chain(hd.h, c, P)
        assert fc == fcur[c] and fb == fbest[c]
    assert np.array_equal(orc.objective_batch(cur, threads=NCPU), fcur)
    assert np.array_equal(orc.objective_batch(best, threads=NCPU), fbest)
    fit, chain, params = B.sap_best(hd.h, P)
    assert fit == fbest.min() and chain == int(np.argmin(fbest)) and np.array_equal(params, best[chain])


# --------------------------------------------------------------------------------- Simulate
@pytest.mark.parametrize("name,count", [("paper_tiny", 512), ("paper_hpg", 512), ("paper_mtb", 256)])
def test_eval_and_simulate_match_oracle(B, paper_problems, name, count):
    prob = paper_problems(name)
    orc = OP.PaperOracle(prob)
    X = PB.random_paper_params(prob, count, seed=21)
    X[0] = prob.truth
    sched = PB.paper_schedule(4, 4, 10, prob.max_objective)
    with Handle(B, prob, sched) as hd:
        assert np.array_equal(B.sap_eval(hd.h, X), orc.objective_batch(X, threads=NCPU))
        assert B.sap_eval(hd.h, X[:1])[0] == orc.objective(prob.truth)
        assert B.sap_get_info(hd.h)["max_objective"] == prob.max_objective
    for x in X[:6]:
        assert np.array_equal(B.sap_simulate(prob, x), orc.simulate(x))


def test_hand_worked_examples_on_the_gpu(B):
    """Examples C, D and E of tests/golden (the oracle's own pins) through sap_simulate / sap_eval."""
    prob = example_c()
    traj = B.sap_simulate(prob, prob.truth)[0]
    for r in golden_rows("example_c_priority.txt"):
        assert traj[int(r[0])].tolist() == [int(v) for v in r[1:]]
    ref = np.full((1, 9, 3), 255, dtype=np.uint8)
    for r in golden_rows("example_d_objective.txt"):
        if r[0] == "R":
            ref[0, :, int(r[1])] = [int(v) for v in r[2:]]
    probd = example_c(ref)
    sched = PB.paper_schedule(2, 2, 5, probd.max_objective)
    with Handle(B, probd, sched) as hd:
        assert B.sap_eval(hd.h, probd.truth)[0] == 15
    src, dst = np.array([0, 1, 2], dtype=np.int32), np.array([1, 2, 0], dtype=np.int32)
    x = np.array([1, 1, 1, 1, -1, 1, 1, 1, 1, 1, 3, 1, 0, 1, 0, 1, 1, 2], dtype=np.int8)
    pe = PB.PaperProblem(name="example_e", seed=0, n_nodes=3, n_edges=3, edge_src=src, edge_dst=dst,
                         fast=np.zeros(3, dtype=np.uint8), n_cond=1, n_steps=7,
                         init_state=np.array([[2, 0, 2]], dtype=np.uint8), ref=np.full((1, 8, 3), 255, dtype=np.uint8))
    traj = B.sap_simulate(pe, x)[0]
    for r in golden_rows("example_e_memory.txt"):
        assert traj[int(r[0])].tolist() == [int(v) for v in r[1:]]


# --------------------------------------------------------------------------------- initial vectors
@pytest.mark.parametrize("name,R", [("paper_tiny", 37), ("paper_hpg", 300), ("paper_mtb", 130)])
@pytest.mark.parametrize("flags", [0, 1])
def test_initial_vectors(B, paper_problems, name, R, flags):
    prob = paper_problems(name)
    orc = OP.PaperOracle(prob)
    sched = PB.paper_schedule(R, 4, 10, prob.max_objective, chain_id_base=5)
    with Handle(B, prob, sched, flags) as hd:
        fcur, fbest = B.sap_get_fitness(hd.h, R)
        for c in range(R):
            x, f = orc.init_chain(sched.seed, c + 5, constrained=bool(flags))
            cur, fc, best, fb = B.sap_get_chain(hd.h, c, prob.n_params)
            assert np.array_equal(cur, x) and np.array_equal(best, x), c
            assert fc == fb == f == fcur[c] == fbest[c], c
            assert not flags or orc.valid(cur)


# --------------------------------------------------------------------------------- chains
@pytest.mark.parametrize("flags", [0, 1])
def test_paper_tiny_full_parity(B, paper_problems, flags):
    prob = paper_problems("paper_tiny")
    orc = OP.PaperOracle(prob)
    spec = PB.PAPER_CONFIGS["paper_tiny"]
    sched = PB.paper_schedule(spec.n_chains, 40, 50, prob.max_objective)
    with Handle(B, prob, sched, flags) as hd:
        chains = list(range(spec.n_chains))
        B.sap_set_trace(hd.h, chains, 2000)
        B.sap_run(hd.h, 700)
        B.sap_run(hd.h, 1300)
        check_chains(B, hd, orc, chains, 2000, B.sap_get_trace(hd.h, len(chains), 2000))
        check_all_fitness(B, hd, orc)


@pytest.mark.parametrize("flags", [0, 1])
def test_paper_hpg_parity(B, paper_problems, flags):
    prob = paper_problems("paper_hpg")
    orc = OP.PaperOracle(prob)
    R = 1000                                                  # not a multiple of the 4 chains a warp carries
    sched = PB.paper_schedule(R, 30, 100, prob.max_objective)
    chains = sorted(set(list(range(0, R, 17)) + [1, 2, 3, R - 3, R - 2, R - 1]))
    with Handle(B, prob, sched, flags) as hd:
        assert B.sap_get_info(hd.h)["lanes_per_chain"] == 8
        B.sap_set_trace(hd.h, chains, 3000)
        B.sap_run(hd.h, 3000)
        check_chains(B, hd, orc, chains, 3000, B.sap_get_trace(hd.h, len(chains), 3000))
        check_all_fitness(B, hd, orc)


@pytest.mark.parametrize("flags", [0, 1])
def test_paper_mtb_parity(B, paper_problems, flags):
    prob = paper_problems("paper_mtb")
    orc = OP.PaperOracle(prob)
    R = 600
    sched = PB.paper_schedule(R, 20, 100, prob.max_objective)
    chains = sorted(set(list(range(0, R, 41)) + [1, 2, 3, R - 1]))
    with Handle(B, prob, sched, flags) as hd:
        assert B.sap_get_info(hd.h)["lanes_per_chain"] == 32
        B.sap_set_trace(hd.h, chains, 2000)
        B.sap_run(hd.h, 2000)
        check_chains(B, hd, orc, chains, 2000, B.sap_get_trace(hd.h, len(chains), 2000))
        check_all_fitness(B, hd, orc)
    # every chain of a full-size launch: the first steps
    spec = PB.PAPER_CONFIGS["paper_mtb"]
    sched = PB.paper_schedule(spec.n_chains, 20, 100, prob.max_objective)
    with Handle(B, prob, sched, flags) as hd:
        B.sap_run(hd.h, 12)
        check_chains(B, hd, orc, list(range(0, spec.n_chains, 16)), 12)


def test_split_runs_and_chain_base(B, paper_problems):
    prob = paper_problems("paper_hpg")
    sched = PB.paper_schedule(24, 10, 50, prob.max_objective)
    with Handle(B, prob, sched, 1) as a:
        B.sap_set_trace(a.h, list(range(24)), 500)
        B.sap_run(a.h, 500)
        ta = B.sap_get_trace(a.h, 24, 500)
    with Handle(B, prob, sched, 1) as b:                                # run(a); run(b) == run(a+b)
        B.sap_set_trace(b.h, list(range(24)), 500)
        for part in (1, 99, 150, 250):
            B.sap_run(b.h, part)
        assert np.array_equal(B.sap_get_trace(b.h, 24, 500), ta)
    part = copy.copy(sched); part.n_chains = 5; part.chain_id_base = 11
    with Handle(B, prob, part, 1) as c:                                 # chain-range partition (reading 25)
        B.sap_set_trace(c.h, [0, 1, 2, 3, 4], 500)
        B.sap_run(c.h, 500)
        assert np.array_equal(B.sap_get_trace(c.h, 5, 500), ta[11:16])
    for env in ({"TSA_PAPER_WPB": "1"}, {"TSA_PAPER_WPB": "8"}, {"TSA_PAPER_LPC": "16"}, {"TSA_PAPER_LPC": "32"}):
        os.environ.update(env)                                          # launch geometry never changes results
        try:
            with Handle(B, prob, sched, 1) as d:
                B.sap_set_trace(d.h, list(range(24)), 500)
                B.sap_run(d.h, 500)
                assert np.array_equal(B.sap_get_trace(d.h, 24, 500), ta), env
        finally:
            for k in env:
                del os.environ[k]


def test_extreme_tables(B, paper_problems):
    prob = paper_problems("paper_hpg")
    orc = OP.PaperOracle(prob)
    greedy = PB.paper_schedule(8, 4, 100, 64)
    greedy.accept = np.zeros_like(greedy.accept)
    hot = PB.paper_schedule(8, 4, 100, prob.max_objective)
    hot.accept = np.full_like(hot.accept, 0xFFFFFFFF)
    for sched in (greedy, hot):
        with Handle(B, prob, sched, 1) as hd:
            B.sap_set_trace(hd.h, list(range(8)), 500)
            B.sap_run(hd.h, 500)                                        # 100 steps past the schedule: the level saturates
            check_chains(B, hd, orc, list(range(8)), 500, B.sap_get_trace(hd.h, 8, 500))


# --------------------------------------------------------------------------------- Table 1 levels
@pytest.mark.parametrize("name,R,levels,spl,group,flags", [("paper_tiny", 8, 10, 20, 0, 0), ("paper_hpg", 96, 5, 40, 0, 1),
                                                           ("paper_hpg", 96, 5, 40, 32, 1), ("paper_mtb", 40, 3, 30, 7, 1)])
def test_run_levels_matches_the_oracle(B, paper_problems, name, R, levels, spl, group, flags):
    prob = paper_problems(name)
    orc = OP.PaperOracle(prob)
    sched = PB.paper_schedule(R, levels, spl, prob.max_objective)
    want = OP.run_levels(orc, sched, R, levels, group, threads=NCPU, constrained=bool(flags))
    with Handle(B, prob, sched, flags) as hd:
        B.sap_run_levels(hd.h, levels, group)
        for c in range(R):
            cur, fc, best, fb = B.sap_get_chain(hd.h, c, prob.n_params)
            assert np.array_equal(cur, want[c][0]) and np.array_equal(best, want[c][1]), c
            assert (fc, fb) == (want[c][2], want[c][3]), c


# --------------------------------------------------------------------------------- acceptance statistics
def test_level_statistics_on_the_device(B, paper_problems):
    """worse solutions accepted per temperature level.  The device counters equal the
    statistics of the traced records of the same run and those of the oracle's traces."""
    prob = paper_problems("paper_hpg")
    orc = OP.PaperOracle(prob)
    R, L, spl = 50, 6, 60
    sched = PB.paper_schedule(R, L, spl, prob.max_objective, t0=30.0, rho=0.6)
    n = L * spl + 45                                                    # 45 steps past the schedule
    with Handle(B, prob, sched, B.SAP_CONSTRAINED | B.SAP_LEVEL_STATS) as hd:
        f0, _ = B.sap_get_fitness(hd.h, R)
        B.sap_set_trace(hd.h, list(range(R)), n)
        B.sap_run(hd.h, 100)
        B.sap_run(hd.h, n - 100)
        got = B.sap_get_level_stats(hd.h, L)
        tr = B.sap_get_trace(hd.h, R, n)
    from_trace = acceptance_by_level(tr, f0, spl, L)
    runs = oracle_chains(orc, sched, list(range(R)), n, True)
    ref = acceptance_by_level(np.stack([r["trace"] for r in runs]), [r["init_fit"] for r in runs], spl, L)
    for k in ("steps", "accepted", "accepted_worse", "improved"):
        assert np.array_equal(got[k], from_trace[k]), k
        assert np.array_equal(got[k], ref[k]), k
    assert got["steps"].sum() == R * n and got["accepted_worse"][0] > got["accepted_worse"][-1]
    with Handle(B, prob, sched, 0) as hd:
        with pytest.raises(B.SaError):
            B.sap_get_level_stats(hd.h, L)


# --------------------------------------------------------------------------------- shapes
SHAPES = [
    # name, N, E, measured, fast, K, T
    ("two_nodes", 2, 2, 1, 1, 1, 1),
    ("lpc16", 20, 55, 11, 6, 2, 7),
    ("four_slots", 100, 320, 56, 30, 1, 12),
    ("eight_slots", 250, 700, 100, 80, 1, 6),
    ("long_course", 12, 30, 7, 4, 1, 300),
]


@pytest.mark.parametrize("shape", SHAPES, ids=[s[0] for s in SHAPES])
def test_edge_shapes(B, shape):
    name, N, E, nm, nf, K, T = shape
    spec = PB.PaperSpec(name, 77, N, E, nm, nf, K, T, 0.05, 16, 200)
    prob = PB.make_paper_problem(name, OP.simulate_fn, spec=spec)
    orc = OP.PaperOracle(prob)
    X = PB.random_paper_params(prob, 64, seed=5)
    sched = PB.paper_schedule(21, 5, 20, min(prob.max_objective, 400))
    for flags in (0, 1):
        with Handle(B, prob, sched, flags) as hd:
            assert np.array_equal(B.sap_eval(hd.h, X), orc.objective_batch(X, threads=NCPU))
            chains = [0, 1, 9, 20]
            B.sap_set_trace(hd.h, chains, 100)
            B.sap_run(hd.h, 100)
            check_chains(B, hd, orc, chains, 100, B.sap_get_trace(hd.h, len(chains), 100))
    assert np.array_equal(B.sap_simulate(prob, X[3]), orc.simulate(X[3]))


def test_source_node_and_validation(B):
    """A node without in-edges has image 0 (it decays); with constraints on the library refuses the
    network (no valid vector exists)."""
    src = np.array([0, 0, 1], dtype=np.int32)
    dst = np.array([1, 2, 2], dtype=np.int32)
    prob = PB.PaperProblem(name="source", seed=0, n_nodes=3, n_edges=3, edge_src=src, edge_dst=dst,
                           fast=np.array([0, 1, 0], dtype=np.uint8), n_cond=1, n_steps=5,
                           init_state=np.array([[2, 1, 0]], dtype=np.uint8), ref=np.full((1, 6, 3), 255, dtype=np.uint8))
    prob.ref[0, :, 2] = [0, 1, 2, 2, 1, 0]
    orc = OP.PaperOracle(prob)
    X = PB.random_paper_params(prob, 200, seed=1)
    sched = PB.paper_schedule(4, 2, 10, 36)
    with Handle(B, prob, sched, 0) as hd:
        assert np.array_equal(B.sap_eval(hd.h, X), orc.objective_batch(X))
        B.sap_set_trace(hd.h, [0, 1, 2, 3], 60)
        B.sap_run(hd.h, 60)
        check_chains(B, hd, orc, [0, 1, 2, 3], 60, B.sap_get_trace(hd.h, 4, 60))
        with pytest.raises(B.SaError):
            bad = X[:1].copy(); bad[0, 0] = 3
            B.sap_eval(hd.h, bad)
    with pytest.raises(B.SaError):
        B.sap_create(prob, sched, B.SAP_CONSTRAINED)


# ------------------------------------------------- the geometry the paper_mtb throughput is measured on
# From R >= 4736 the planner gives paper_mtb 16 lanes per chain: two chains per warp, four node slots per lane
# (sap_plan.cpp).  The long-trace tests above run the 32-lane geometry, so this one gets its own: forced at a small R,
# then chosen by the planner at the benchmark's R, odd and even chains (the second and the first chain of a warp).
@pytest.mark.parametrize("flags", [0, 1])
def test_paper_mtb_two_chains_per_warp_forced(B, paper_problems, flags):
    prob = paper_problems("paper_mtb")
    orc = OP.PaperOracle(prob)
    R = 601                                                   # odd: the last warp carries one chain only
    sched = PB.paper_schedule(R, 20, 100, prob.max_objective)
    chains = sorted(set(list(range(0, R, 29)) + list(range(1, R, 31)) + [2, 3, R - 2, R - 1]))
    assert len(chains) >= 40 and sum(c & 1 for c in chains) >= 15 and sum(1 - (c & 1) for c in chains) >= 15
    os.environ["TSA_PAPER_LPC"] = "16"
    try:
        with Handle(B, prob, sched, flags) as hd:
            assert B.sap_get_info(hd.h)["lanes_per_chain"] == 16
            B.sap_set_trace(hd.h, chains, 2000)
            B.sap_run(hd.h, 700)
            B.sap_run(hd.h, 1300)
            check_chains(B, hd, orc, chains, 2000, B.sap_get_trace(hd.h, len(chains), 2000))
            check_all_fitness(B, hd, orc)
    finally:
        del os.environ["TSA_PAPER_LPC"]


@pytest.mark.parametrize("flags", [0, 1])
def test_paper_mtb_benchmarked_geometry_full_length(B, paper_problems, flags):
    prob = paper_problems("paper_mtb")
    orc = OP.PaperOracle(prob)
    spec = PB.PAPER_CONFIGS["paper_mtb"]
    R, steps = spec.n_chains, spec.sa_steps                   # 10 240 chains x 5000 steps, as bench.py runs it
    sched = PB.paper_schedule(R, 50, steps // 50, prob.max_objective)
    chains = sorted(set(list(range(0, R, 331)) + list(range(1, R, 641)) + [R - 2, R - 1]))
    assert len(chains) >= 32 and sum(c & 1 for c in chains) >= 10
    with Handle(B, prob, sched, flags) as hd:
        assert B.sap_get_info(hd.h)["lanes_per_chain"] == 16  # the planner's own choice at this R
        B.sap_set_trace(hd.h, chains, steps)
        B.sap_run(hd.h, 12)
        check_chains(B, hd, orc, list(range(R)), 12)          # every chain, not every 16th
        B.sap_run(hd.h, steps - 12)
        check_chains(B, hd, orc, chains, steps, B.sap_get_trace(hd.h, len(chains), steps))
        check_all_fitness(B, hd, orc)


def test_paper_mtb_hundred_thousand_chains(B, paper_problems):
    prob = paper_problems("paper_mtb")
    orc = OP.PaperOracle(prob)
    R = 102400
    sched = PB.paper_schedule(R, 4, 5, prob.max_objective)
    with Handle(B, prob, sched, 1) as hd:
        assert B.sap_get_info(hd.h)["lanes_per_chain"] == 16
        B.sap_run(hd.h, 20)
        check_chains(B, hd, orc, list(range(0, R, 7)) + [R - 1], 20)


# ------------------------------------------------------------------------------------- autoregulation
def with_self_loops(prob, count=6):
    """A copy of the problem in which `count` edges are turned into self-loops (src -> src).  Only edges whose target
    keeps at least two other in-edges are taken, so that every node still has an in-edge and an out-edge."""
    src, dst = prob.edge_src.copy(), prob.edge_dst.copy()
    have = set(zip(src.tolist(), dst.tolist()))
    indeg = np.bincount(dst, minlength=prob.n_nodes)
    done = 0
    for e in range(prob.n_edges):
        s, d = int(src[e]), int(dst[e])
        if done < count and indeg[d] >= 3 and (s, s) not in have:
            have.discard((s, d)); have.add((s, s))
            indeg[d] -= 1; indeg[s] += 1
            dst[e] = s
            done += 1
    assert done == count
    out = copy.copy(prob)
    out.edge_src, out.edge_dst = src, dst
    return out


@pytest.mark.parametrize("name,R,flags", [("paper_hpg", 64, 0), ("paper_hpg", 64, 1), ("paper_mtb", 48, 1), ("paper_mtb", 9600, 1)])
def test_self_loops_are_edges_like_any_other(B, paper_problems, name, R, flags):
    prob = with_self_loops(paper_problems(name))
    assert int((prob.edge_src == prob.edge_dst).sum()) == 6
    orc = OP.PaperOracle(prob)
    sched = PB.paper_schedule(R, 10, 80, prob.max_objective)
    chains = PB.spread_chains(R, 24)
    with Handle(B, prob, sched, flags) as hd:
        B.sap_set_trace(hd.h, chains, 800)
        B.sap_run(hd.h, 800)
        tr = B.sap_get_trace(hd.h, len(chains), 800)
        check_chains(B, hd, orc, chains, 800, tr)
        loops = np.nonzero(prob.edge_src == prob.edge_dst)[0]
        param = OP.unpack_trace(tr)["param"]                             # weight, polarity and threshold of edge e: e, E + e, 2E + e
        assert np.isin(param[param < 3 * prob.n_edges] % prob.n_edges, loops).any(), "no self-loop parameter was ever proposed"
        x = PB.random_paper_params(prob, 64, 5)
        assert np.array_equal(B.sap_eval(hd.h, x), orc.objective_batch(x))
        assert np.array_equal(B.sap_simulate(prob, x[0]), orc.simulate(x[0]))


def test_set_trace_refuses_sizes_that_cannot_be_a_buffer(B, paper_problems):
    prob = paper_problems("paper_tiny")
    sched = PB.paper_schedule(8, 4, 25, prob.max_objective)
    with Handle(B, prob, sched) as hd:
        for n, steps in ((2, 2 ** 62), (8, 2 ** 61), (1, 2 ** 34 + 1)):
            with pytest.raises(B.SaError) as err:
                B.sap_set_trace(hd.h, list(range(n)), steps)
            assert err.value.code == B.SA_EINVAL and "trace records" in str(err.value)
        B.sap_set_trace(hd.h, [5], 40)
        B.sap_run(hd.h, 40)
        check_chains(B, hd, OP.PaperOracle(prob), [5], 40, B.sap_get_trace(hd.h, 1, 40))
