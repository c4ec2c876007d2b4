"""Parity of the CUDA path (through the C ABI) against the CPU oracle — bit-exact, element by
element, on the same seeded inputs.  Everything here needs a GPU (-m gpu)."""
import copy
import os
from concurrent.futures import ThreadPoolExecutor

import numpy as np
import pytest

from oracle import oracle as O
from paper_2506_19866_b200 import problems as PB
from helpers import all_settings, brute_force_problem, example_problem

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


class Handle:
    def __init__(self, B, prob, sched):
        self.B, self.prob, self.sched = B, prob, sched
        self.h = B.sa_create(prob, sched)

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.B.sa_destroy(self.h)


def oracle_chains(orc, sched, chains, n_steps):
    with ThreadPoolExecutor(NCPU) as ex:
        return list(ex.map(lambda c: orc.run_chain(sched, c + sched.chain_id_base, n_steps), chains))


def check_chains(B, hd, orc, chains, n_steps, trace=None):
    """GPU state of `chains` after n_steps from a fresh handle == oracle (trace, vectors, fitness)."""
    refs = oracle_chains(orc, hd.sched, chains, n_steps)
    for row, (c, ref) in enumerate(zip(chains, refs)):
        cur, fc, best, fb = B.sa_get_chain(hd.h, c, hd.prob.n_params)
        if trace is not None:
            bad = np.nonzero(trace[row][:n_steps] != ref["trace"])[0]
            assert bad.size == 0, f"chain {c}: first trace mismatch at step {bad[0]}: " \
                                  f"gpu {int(trace[row][bad[0]]):#x} oracle {int(ref['trace'][bad[0]]):#x}"
        assert (fc, fb) == (ref["fit_cur"], ref["fit_best"]), f"chain {c} fitness"
        assert np.array_equal(cur, ref["cur"]), f"chain {c} current vector"
        assert np.array_equal(best, ref["best"]), f"chain {c} best vector"


def check_all_fitness(B, hd, orc):
    """For every chain: reported d_cur / d_best equal the ORACLE fitness of the returned vectors."""
    R, P = hd.sched.n_chains, hd.prob.n_params
    fcur, fbest = B.sa_get_fitness(hd.h, R)
    assert (fbest <= fcur).all()
    cur = np.zeros((R, P), dtype=np.int8)
    best = np.zeros((R, P), dtype=np.int8)
    for c in range(R):
        cur[c], fc, best[c], fb = B.sa_get_chain(hd.h, c, P)
        assert fc == fcur[c] and fb == fbest[c]
    assert np.array_equal(orc.fitness_batch(cur, threads=NCPU), fcur)
    assert np.array_equal(orc.fitness_batch(best, threads=NCPU), fbest)
    fit, chain, params = B.sa_best(hd.h, P)
    assert fit == fbest.min() and chain == int(np.argmin(fbest)) and np.array_equal(params, best[chain])


# --------------------------------------------------------------------------------- fitness
@pytest.mark.parametrize("name,count", [("tiny", 256), ("hpg", 256), ("mtb", 128), ("large", 12)])
def test_eval_and_simulate_match_oracle(B, problems_cache, name, count):
    prob = problems_cache(name)
    orc = O.Oracle(prob)
    assert np.array_equal(B.sa_simulate(prob, prob.truth), orc.states_at_obs(prob.truth))
    X = np.concatenate([PB.random_params(prob, count, seed=21), prob.truth[None, :]])
    with Handle(B, prob, PB.default_schedule(name, n_chains=4)) as hd:
        got = B.sa_eval(hd.h, X)
    want = orc.fitness_batch(X, threads=NCPU)
    assert np.array_equal(got, want)
    assert got[-1] == prob.n_flipped


def test_eval_hand_worked_examples(B):
    prob = example_problem(with_condition_b=True)
    sched = PB.make_schedule(2, 100)
    X = np.stack([prob.truth] * 4)
    X[1, 0] = 0; X[2, 7] = 5; X[3, 4] = 1
    with Handle(B, prob, sched) as hd:
        assert B.sa_eval(hd.h, X).tolist() == [1, 2, 5, 2]          # tests/golden/example_b_fitness.txt
    probA = example_problem()
    assert np.array_equal(B.sa_simulate(probA, probA.truth), O.Oracle(probA).states_at_obs(probA.truth))


def test_eval_brute_force_every_setting(B):
    prob = brute_force_problem(O.simulate_fn)
    X = all_settings(6, 4, 6)
    want = O.Oracle(prob).fitness_batch(X, threads=NCPU)
    with Handle(B, prob, PB.make_schedule(2, 100)) as hd:
        got = B.sa_eval(hd.h, X)
    assert np.array_equal(got, want)                                # all 944 784 elements


# --------------------------------------------------------------------------------- SA runs
def test_tiny_full_parity(B, problems_cache):
    prob = problems_cache("tiny")
    sched = PB.default_schedule("tiny")
    orc = O.Oracle(prob)
    chains = list(range(8))
    with Handle(B, prob, sched) as hd:
        f0, _ = B.sa_get_fitness(hd.h, 8)
        assert f0.tolist() == [orc.init_chain(sched.seed, c)[1] for c in chains]
        B.sa_set_trace(hd.h, chains, 2000)
        B.sa_run(hd.h, 2000)
        check_chains(B, hd, orc, chains, 2000, B.sa_get_trace(hd.h, 8, 2000))
        check_all_fitness(B, hd, orc)


def test_hpg_full_size_parity(B, problems_cache):
    """HPG-shaped, ALL 1024 chains x 20 000 steps, full trace."""
    prob = problems_cache("hpg")
    sched = PB.default_schedule("hpg")                                # R = 1024, 20 000 steps
    orc = O.Oracle(prob)
    chains = list(range(1024))
    with Handle(B, prob, sched) as hd:
        B.sa_set_trace(hd.h, chains, 20000)
        B.sa_run(hd.h, 20000)
        check_chains(B, hd, orc, chains, 20000, B.sa_get_trace(hd.h, len(chains), 20000))
        check_all_fitness(B, hd, orc)


def test_mtb_full_size_parity(B, problems_cache):
    """Mtb-shaped, 32 chains (0-3 and 28 evenly spread) x 20 000 steps with trace; all
    4096 chains x the first 20 steps."""
    prob = problems_cache("mtb")
    sched = PB.default_schedule("mtb")                                # R = 4096, 20 000 steps
    orc = O.Oracle(prob)
    chains = sorted(set(PB.spread_chains(4096, 32) + [4095]))
    assert len(chains) >= 32
    with Handle(B, prob, sched) as hd:
        B.sa_set_trace(hd.h, chains, 20000)
        B.sa_run(hd.h, 20000)
        check_chains(B, hd, orc, chains, 20000, B.sa_get_trace(hd.h, len(chains), 20000))
        check_all_fitness(B, hd, orc)
    with Handle(B, prob, sched) as hd:                                # every chain, first 20 steps
        f0, _ = B.sa_get_fitness(hd.h, 4096)
        B.sa_run(hd.h, 20)
        refs = oracle_chains(orc, sched, list(range(4096)), 20)
        assert f0.tolist() == [r["init_fit"] for r in refs]
        check_chains(B, hd, orc, list(range(4096)), 20)


def test_scaling_chain_counts(B, problems_cache):
    """per R 8 spread chains x 2000 steps, all chains x 2 steps, and chain c identical
    across the three R (invariant vii)."""
    prob = problems_cache("mtb")
    orc = O.Oracle(prob)
    common = [0, 1, 500, 1023]
    traces = {}
    for R in PB.SCALING_CHAINS:
        sched = PB.default_schedule("mtb", n_chains=R, total_steps=PB.SCALING_STEPS)
        chains = sorted(set(common + PB.spread_chains(R, 8)))
        with Handle(B, prob, sched) as hd:
            B.sa_set_trace(hd.h, chains, 2000)
            B.sa_run(hd.h, 2000)
            tr = B.sa_get_trace(hd.h, len(chains), 2000)
            check_chains(B, hd, orc, chains, 2000, tr)
            traces[R] = {c: tr[chains.index(c)] for c in common}
            if R == 1024:
                check_all_fitness(B, hd, orc)
        with Handle(B, prob, sched) as hd:                            # all chains x 2 steps
            B.sa_run(hd.h, 2)
            check_chains(B, hd, orc, list(range(R)), 2)
    for c in common:                                                  # invariant (vii): independent of R
        assert np.array_equal(traces[1024][c], traces[8192][c]) and np.array_equal(traces[1024][c], traces[65536][c])


def test_large_parity(B, problems_cache):
    """Large, 8 chains x 1000 steps with trace; all 2048 chains: initial fitness + 1 step."""
    prob = problems_cache("large")
    sched = PB.default_schedule("large")                              # R = 2048, 1000 steps
    orc = O.Oracle(prob)
    chains = PB.spread_chains(2048, 8)
    with Handle(B, prob, sched) as hd:
        f0, _ = B.sa_get_fitness(hd.h, 2048)
        with ThreadPoolExecutor(NCPU) as ex:
            want0 = list(ex.map(lambda c: orc.init_chain(sched.seed, c)[1], range(2048)))
        assert f0.tolist() == want0                                   # all chains: initial fitness
        B.sa_set_trace(hd.h, chains, 1000)
        B.sa_run(hd.h, 1000)
        check_chains(B, hd, orc, chains, 1000, B.sa_get_trace(hd.h, len(chains), 1000))
    with Handle(B, prob, sched) as hd:                                # all chains: one step
        B.sa_run(hd.h, 1)
        check_chains(B, hd, orc, list(range(2048)), 1)


# --------------------------------------------------------------------------------- invariants
def test_split_runs_chain_base_and_team_width(B, problems_cache):
    prob = problems_cache("mtb")
    sched = PB.default_schedule("mtb", n_chains=16, total_steps=600)
    with Handle(B, prob, sched) as a:
        B.sa_set_trace(a.h, list(range(16)), 600)
        B.sa_run(a.h, 600)
        ta = B.sa_get_trace(a.h, 16, 600)
        state_a = [B.sa_get_chain(a.h, c, prob.n_params) for c in range(16)]
    with Handle(B, prob, sched) as b:                                 # run(a); run(b) == run(a+b)
        B.sa_set_trace(b.h, list(range(16)), 600)
        for part in (1, 99, 250, 250):
            B.sa_run(b.h, part)
        assert np.array_equal(B.sa_get_trace(b.h, 16, 600), ta)
    part_sched = copy.copy(sched); part_sched.n_chains = 4; part_sched.chain_id_base = 8
    with Handle(B, prob, part_sched) as c:                            # chain-range partition (reading 25)
        B.sa_set_trace(c.h, [0, 1, 2, 3], 600)
        B.sa_run(c.h, 600)
        assert np.array_equal(B.sa_get_trace(c.h, 4, 600), ta[8:12])
    # launch geometry and the host's edge schedule never change results
    for env in ({"TSA_TEAM_WARPS": "1"}, {"TSA_TEAM_WARPS": "2"}, {"TSA_TEAM_WARPS": "4"},
                {"TSA_NO_SPLIT": "1"}, {"TSA_NO_BANKOPT": "1"}, {"TSA_NO_SPLIT": "1", "TSA_NO_BANKOPT": "1"}):
        os.environ.update(env)
        try:
            with Handle(B, prob, sched) as d:
                B.sa_select_kernel(d.h, B.SA_KERNEL_GENERIC if "TSA_TEAM_WARPS" in env else B.SA_KERNEL_STATIC)
                info = B.sa_get_info(d.h)
                if "TSA_TEAM_WARPS" in env:
                    assert info["threads_per_cta"] == 32 * int(env["TSA_TEAM_WARPS"])
                if "TSA_NO_SPLIT" in env:
                    assert info["split_nodes"] == 0
                B.sa_run(d.h, 600)
                for ch in range(16):
                    got = B.sa_get_chain(d.h, ch, prob.n_params)
                    assert np.array_equal(got[0], state_a[ch][0]) and got[1] == state_a[ch][1]
                    assert np.array_equal(got[2], state_a[ch][2]) and got[3] == state_a[ch][3]
        finally:
            for k in env:
                del os.environ[k]


FAMILY_CASES = [
    # problem, family, environment
    ("hpg", "GENERIC", {}), ("hpg", "STATIC", {}), ("hpg", "DENSE", {}),
    ("mtb", "GENERIC", {}), ("mtb", "STATIC", {}), ("mtb", "DENSE", {}),
    ("mtb", "DENSE", {"TSA_DENSE_W": "2"}), ("mtb", "DENSE", {"TSA_DENSE_W": "4"}),
    ("mtb", "DENSE", {"TSA_DENSE_BLOCKS": "8"}), ("mtb", "DENSE", {"TSA_DENSE_PH": "2"}),
    ("mtb", "DENSE", {"TSA_DENSE_CPB": "8"}), ("mtb", "DENSE", {"TSA_DENSE_CPB": "12"}), ("mtb", "DENSE", {"TSA_DENSE_CPB": "16"}),
    ("hpg", "DENSE", {"TSA_DENSE_CPB": "4"}),
    ("mtb", "DENSE", {"TSA_DENSE_SP": "0"}), ("mtb", "DENSE", {"TSA_DENSE_SP": "0", "TSA_DENSE_W": "2"}),
    ("mtb", "DENSE", {"TSA_DENSE_SP": "0", "TSA_DENSE_CPB": "8"}),
    # round 2: register exchange through movmatrix, thresholds folded into the C operand, chains per CTA
    ("mtb", "DENSE", {"TSA_DENSE_MOVM": "1"}), ("hpg", "DENSE", {"TSA_DENSE_MOVM": "1"}),
    ("mtb", "DENSE", {"TSA_DENSE_MOVM": "1", "TSA_DENSE_SP": "0"}), ("mtb", "DENSE", {"TSA_DENSE_MOVM": "1", "TSA_DENSE_CPB": "16"}),
    ("mtb", "DENSE", {"TSA_DENSE_CFOLD": "1"}), ("hpg", "DENSE", {"TSA_DENSE_CFOLD": "0"}), ("hpg", "DENSE", {"TSA_DENSE_CFOLD": "1", "TSA_DENSE_MOVM": "1"}),
    ("mtb", "DENSE", {"TSA_DENSE_CPB": "1"}), ("mtb", "DENSE", {"TSA_DENSE_CPB": "7"}),
    # speculative look-ahead: 2 .. 4 warps per chain score consecutive SA steps at once
    ("hpg", "DENSE", {"TSA_DENSE_SPEC": "2"}), ("hpg", "DENSE", {"TSA_DENSE_SPEC": "3", "TSA_DENSE_CPB": "7"}),
    ("hpg", "DENSE", {"TSA_DENSE_SPEC": "4", "TSA_DENSE_CPB": "4"}), ("mtb", "DENSE", {"TSA_DENSE_SPEC": "2", "TSA_DENSE_CPB": "8"}),
    ("mtb", "DENSE", {"TSA_DENSE_SPEC": "3", "TSA_DENSE_SP": "0"}), ("hpg", "DENSE", {"TSA_DENSE_SPEC": "2", "TSA_DENSE_MOVM": "1"}),
]


@pytest.mark.parametrize("name,family,env", FAMILY_CASES, ids=[f"{n}-{f}-{'-'.join(k[10:] + v for k, v in e.items()) or 'default'}" for n, f, e in FAMILY_CASES])
def test_every_kernel_family_matches_the_oracle(B, problems_cache, name, family, env):
    """sa_run has three kernel families (include/ternary_sa.h); each one, forced, reproduces the
    oracle's trace, vectors and fitness, and says which one ran."""
    prob = problems_cache(name)
    orc = O.Oracle(prob)
    sched = PB.default_schedule(name, n_chains=24, total_steps=400)
    chains = [0, 1, 7, 23]
    os.environ.update(env)
    try:
        with Handle(B, prob, sched) as hd:
            B.sa_select_kernel(hd.h, getattr(B, "SA_KERNEL_" + family))
            B.sa_set_trace(hd.h, chains, 400)
            B.sa_run(hd.h, 130)
            B.sa_run(hd.h, 270)
            info = B.sa_get_info(hd.h)
            assert info["variant"] == {"GENERIC": info["variant"], "STATIC": 4, "DENSE": 5}[family]
            assert family != "GENERIC" or info["variant"] in (2, 3)
            if "TSA_DENSE_W" in env:
                assert info["threads_per_cta"] == 32 * int(env["TSA_DENSE_W"])
            check_chains(B, hd, orc, chains, 400, B.sa_get_trace(hd.h, len(chains), 400))
            check_all_fitness(B, hd, orc)
    finally:
        for k in env:
            del os.environ[k]


def test_balanced_slots_hand_chains_over(B, problems_cache):
    """More chains than resident slots: the dense kernel splits the line of R*steps chain-steps evenly
    over the slots and hands straddling chains from one slot to the next through HBM.  Results are
    those of the plain launch and of the oracle; two sa_run calls cut the line at different places."""
    prob = problems_cache("mtb")
    orc = O.Oracle(prob)
    R, steps = 2600, 44
    sched = PB.default_schedule("mtb", n_chains=R, total_steps=steps)
    chains = sorted(set(list(range(0, R, 113)) + [1, 2, 3, R - 2, R - 1]))
    with Handle(B, prob, sched) as hd:
        B.sa_select_kernel(hd.h, B.SA_KERNEL_DENSE)
        B.sa_set_trace(hd.h, chains, steps)
        B.sa_run(hd.h, 17)
        B.sa_run(hd.h, steps - 17)
        info = B.sa_get_info(hd.h)
        assert info["variant"] == 5 and info["grid"] * info["chains_per_cta"] < R, info
        check_chains(B, hd, orc, chains, steps, B.sa_get_trace(hd.h, len(chains), steps))
        balanced = B.sa_get_fitness(hd.h, R)
    os.environ["TSA_DENSE_NO_BALANCE"] = "1"
    try:
        with Handle(B, prob, sched) as hd:
            B.sa_select_kernel(hd.h, B.SA_KERNEL_DENSE)
            B.sa_run(hd.h, steps)
            info = B.sa_get_info(hd.h)
            assert info["grid"] == -(-R // info["chains_per_cta"]), info       # one chain per slot, no hand-over
            plain = B.sa_get_fitness(hd.h, R)
    finally:
        del os.environ["TSA_DENSE_NO_BALANCE"]
    assert np.array_equal(balanced[0], plain[0]) and np.array_equal(balanced[1], plain[1])


def test_sparse_operand_applies_or_falls_back(B):
    """The 2:4-sparse A operand needs at most two candidate edges per row in every group of four
    columns after the host's node permutation: sparse networks get it, a candidate graph that is 60 %
    full cannot, and AUTO then runs the dense operand.  Same results either way."""
    for name, N, E, want_sparse in (("sp_ok", 60, 420, 1), ("sp_full", 40, 940, 0)):
        cs = PB.ConfigSpec(name, 31 + N, N, E, "uniform-pairs", 6, 2, 8, (4, 8), 8, 150, max_in_degree=39)
        prob = PB.make_problem(name, O.simulate_fn, spec=cs, noise=0.05)
        orc = O.Oracle(prob)
        sched = PB.make_schedule(8, 150)
        with Handle(B, prob, sched) as hd:
            B.sa_select_kernel(hd.h, B.SA_KERNEL_DENSE)
            B.sa_set_trace(hd.h, list(range(8)), 150)
            B.sa_run(hd.h, 150)
            di = B.sa_get_dense_info(hd.h)
            assert di["applies"] == 1 and di["sparse"] == want_sparse, di
            check_chains(B, hd, orc, list(range(8)), 150, B.sa_get_trace(hd.h, 8, 150))


EMPTY_BLOCK_CASES = [("eb100a", 100, 900, "powerlaw", 7), ("eb100b", 100, 700, "poisson", 11), ("eb116", 116, 640, "poisson", 5),
                     ("eb84", 84, 500, "powerlaw", 3), ("eb68", 68, 420, "poisson", 9), ("eb104", 104, 1500, "poisson", 2),
                     ("eb128", 128, 800, "powerlaw", 4), ("eb112", 112, 700, "poisson", 6), ("eb90", 90, 600, "powerlaw", 8)]


@pytest.mark.parametrize("name,N,E,degree,seed", EMPTY_BLOCK_CASES, ids=[c[0] for c in EMPTY_BLOCK_CASES])
def test_empty_blocks_of_the_weight_matrix(B, name, N, E, degree, seed):
    """A last row tile with few nodes: the host tries to number the nodes so that one or two blocks of the weight
    matrix hold no candidate edge (their IMMAs are left out) and falls back to the plain numbering if the pinned
    2:4 search fails.  Whatever it finds, the results are the oracle's."""
    cs = PB.ConfigSpec(name, 4000 + seed, N, E, degree, 8, 3, 16, (4, 8, 12, 16), 8, 120, max_in_degree=40)
    prob = PB.make_problem(name, O.simulate_fn, spec=cs, noise=0.05)
    orc = O.Oracle(prob)
    sched = PB.make_schedule(8, 120)
    with Handle(B, prob, sched) as hd:
        B.sa_select_kernel(hd.h, B.SA_KERNEL_DENSE)
        B.sa_set_trace(hd.h, list(range(8)), 120)
        B.sa_run(hd.h, 120)
        di = B.sa_get_dense_info(hd.h)
        blocks = di["row_tiles"] * (di["col_steps"] // 2 if di["sparse"] else di["col_steps"])
        assert di["applies"] == 1 and 0 < di["immas_per_step"] <= blocks, di
        check_chains(B, hd, orc, list(range(8)), 120, B.sa_get_trace(hd.h, 8, 120))
        check_all_fitness(B, hd, orc)


def test_dense_kernel_limits(B):
    """The dense family applies up to 128 nodes and 8 conditions; beyond that DENSE fails loudly
    and AUTO falls back to the gather kernels with identical results."""
    for name, N, E, K in (("n128", 128, 700, 8), ("n129", 129, 700, 8), ("k9", 40, 160, 9)):
        cs = PB.ConfigSpec(name, 777 + N + K, N, E, "poisson", K, 2, 10, (5, 10), 8, 200, max_in_degree=40)
        prob = PB.make_problem(name, O.simulate_fn, spec=cs, noise=0.05)
        orc = O.Oracle(prob)
        sched = PB.make_schedule(8, 200)
        with Handle(B, prob, sched) as hd:
            B.sa_set_trace(hd.h, list(range(8)), 200)
            B.sa_run(hd.h, 200)
            assert (B.sa_get_info(hd.h)["variant"] == 5) == (name == "n128")
            check_chains(B, hd, orc, list(range(8)), 200, B.sa_get_trace(hd.h, 8, 200))
        if name != "n128":
            with Handle(B, prob, sched) as hd:
                B.sa_select_kernel(hd.h, B.SA_KERNEL_DENSE)
                with pytest.raises(B.SaError):
                    B.sa_run(hd.h, 1)


def test_extreme_tables(B, problems_cache):
    prob = problems_cache("hpg")
    orc = O.Oracle(prob)
    greedy = PB.make_schedule(8, 400)
    greedy.accept = np.zeros_like(greedy.accept)
    hot = PB.make_schedule(8, 400, dmax=prob.n_scored)
    hot.accept = np.full((hot.n_levels, prob.n_scored), 0xFFFFFFFF, dtype=np.uint32)
    for sched in (greedy, hot):
        with Handle(B, prob, sched) as hd:
            B.sa_set_trace(hd.h, list(range(8)), 400)
            B.sa_run(hd.h, 400)
            check_chains(B, hd, orc, list(range(8)), 400, B.sa_get_trace(hd.h, 8, 400))
    # past the end of the schedule the level saturates at L-1 (reading 20)
    short = PB.make_schedule(4, 200, n_levels=10)
    with Handle(B, prob, short) as hd:
        B.sa_set_trace(hd.h, [0, 1, 2, 3], 500)
        B.sa_run(hd.h, 500)
        check_chains(B, hd, orc, [0, 1, 2, 3], 500, B.sa_get_trace(hd.h, 4, 500))


# --------------------------------------------------------------------------------- edge cases
EDGE_SPECS = [
    # name            N   E   degree           K  clamp T  obs_times
    ("k1",            9,  20, "uniform-pairs", 1, 1,    5, (1, 5)),
    ("k5_pad_lanes",  12, 40, "poisson",       5, 2,    7, (2, 4, 7)),
    ("k9",            20, 70, "poisson",       9, 1,    6, (3, 6)),
    ("k17_chunks",    10, 30, "uniform-pairs", 17, 1,   6, (2, 6)),
    ("k37_chunks",    8,  24, "uniform-pairs", 37, 2,   4, (1, 2, 3, 4)),
    ("n33_two_pass",  33, 120, "poisson",      4, 3,    8, (4, 8)),
    ("n70_ragged",    70, 400, "powerlaw",     6, 2,    9, (3, 6, 9)),
    ("t1",            16, 50, "poisson",       3, 1,    1, (1,)),
    ("all_clamped",   6,  12, "uniform-pairs", 2, 6,    4, (2, 4)),
    ("sparse",        40, 41, "uniform-pairs", 8, 1,    10, (5, 10)),
]


@pytest.mark.parametrize("spec", EDGE_SPECS, ids=[s[0] for s in EDGE_SPECS])
def test_edge_shapes(B, spec):
    name, N, E, degree, K, nclamp, T, times = spec
    cs = PB.ConfigSpec(name, 4242 + N + K, N, E, degree, K, nclamp, T, times, 12, 300,
                       max_in_degree=min(N - 1, 40))
    prob = PB.make_problem(name, O.simulate_fn, spec=cs, noise=0.10)
    orc = O.Oracle(prob)
    sched = PB.make_schedule(12, 300)
    X = PB.random_params(prob, 64, seed=N)
    with Handle(B, prob, sched) as hd:
        assert np.array_equal(B.sa_eval(hd.h, X), orc.fitness_batch(X))
        assert np.array_equal(B.sa_simulate(prob, prob.truth), orc.states_at_obs(prob.truth))
        B.sa_set_trace(hd.h, list(range(12)), 300)
        B.sa_run(hd.h, 300)
        check_chains(B, hd, orc, list(range(12)), 300, B.sa_get_trace(hd.h, 12, 300))
        check_all_fitness(B, hd, orc)


def test_nothing_observed_and_max_in_degree(B):
    # nothing observed: fitness is 0 for everything, every move has d = 0 and is accepted
    cs = PB.ConfigSpec("blind", 99, 10, 30, "uniform-pairs", 3, 1, 5, (2, 5), 4, 100)
    prob = PB.make_problem("blind", O.simulate_fn, spec=cs)
    prob.obs = np.full_like(prob.obs, 255)
    sched = PB.make_schedule(4, 100)
    orc = O.Oracle(prob)
    with Handle(B, prob, sched) as hd:
        B.sa_set_trace(hd.h, [0, 1, 2, 3], 100)
        B.sa_run(hd.h, 100)
        tr = B.sa_get_trace(hd.h, 4, 100)
        assert O.unpack_trace(tr)["accepted"].all() and (O.unpack_trace(tr)["delta_cand"] == 0).all()
        check_chains(B, hd, orc, [0, 1, 2, 3], 100, tr)
    # a hub with in-degree 62 (the accumulator limit) fed by nodes stuck at 2: sums reach +-124
    N = 64
    star = copy.copy(prob)
    star.n_nodes, star.n_edges = N, 62 + 1
    star.edge_src = np.array(list(range(1, 63)) + [0], dtype=np.int32)
    star.edge_dst = np.array([0] * 62 + [63], dtype=np.int32)
    star.init_state = np.full((3, N), 2, dtype=np.uint8)
    star.clamp = np.ones((3, N), dtype=np.uint8); star.clamp[:, 0] = 0; star.clamp[:, 63] = 0
    star.obs = np.full((3, 2, N), 255, dtype=np.uint8); star.obs[:, :, 0] = 1; star.obs[:, :, 63] = 2
    orc = O.Oracle(star)
    X = PB.random_params(star, 40, seed=5)
    X[0, :63] = 1; X[1, :63] = -1; X[2, :62] = 1; X[2, 62] = -1
    with Handle(B, star, sched) as hd:
        assert np.array_equal(B.sa_eval(hd.h, X), orc.fitness_batch(X))
        B.sa_run(hd.h, 100)
        check_chains(B, hd, orc, [0, 1, 2, 3], 100)


def test_int32_peak_microbenchmark_runs(B):
    pk = B.sa_int32_peak()
    assert pk["sm_count"] > 0 and pk["sm_hz"] > 2e8
    for k in ("iadd3", "lop3", "imad", "mixed"):
        # never above one instruction per scheduler per clock, never absurdly low
        ceiling = pk["sm_count"] * 4 * pk["sm_hz"]
        assert 0.05 * ceiling < pk[k] < 1.05 * ceiling, (k, pk)


@pytest.mark.gpu
def test_set_trace_refuses_sizes_that_cannot_be_a_buffer(B, problems_cache):
    """chains x steps x 8 bytes is checked before it can wrap or reach the allocator (2^34 records at most)."""
    prob = problems_cache("tiny")
    sched = PB.default_schedule("tiny")
    with Handle(B, prob, sched) as hd:
        for n, steps in ((2, 2 ** 62), (8, 2 ** 61), (1, 2 ** 34 + 1), (8, 2 ** 32)):
            with pytest.raises(B.SaError) as err:
                B.sa_set_trace(hd.h, list(range(n)), steps)
            assert err.value.code == B.SA_EINVAL and "trace records" in str(err.value)
        B.sa_set_trace(hd.h, [0, 3], 50)                                  # and tracing still works afterwards
        B.sa_run(hd.h, 50)
        tr = B.sa_get_trace(hd.h, 2, 50)
        ref = O.Oracle(prob).run_chain(sched, 3, 50)
        assert np.array_equal(tr[1], ref["trace"])
