"""Pins for the CPU oracle (SURVEY.md §8(c) "What pins the oracle"): none of these retypes the
oracle's own formula — they are hand-worked values (tests/golden), closed forms, invariants,
a dense library-matmul special case and brute force on a tiny network."""
import copy
import os

import numpy as np
import pytest

from oracle import oracle as O
from paper_2506_19866_b200 import problems as PB
from helpers import all_settings, aten_philox_blocks, brute_force_problem, example_problem, golden_rows


# ------------------------------------------------------------------ Pin 1 / Pin 2: hand-worked
def test_example_a_trajectory():
    prob = example_problem()
    traj = O.Oracle(prob).simulate(prob.truth)[0]            # [T+1][N]
    rows = golden_rows("example_a_trajectory.txt")
    assert len(rows) == 7
    for r in rows:
        t, want = int(r[0]), [int(v) for v in r[1:]]
        assert traj[t].tolist() == want, f"t={t}"
    # in-place (asynchronous) updating would give node1 = 1 at t=1 (golden header)
    assert traj[1, 1] == 0
    # period 4 from t=2 on: t=6 equals t=2
    assert traj[6].tolist() == traj[2].tolist()


def test_example_b_fitness_and_candidates():
    prob = example_problem(with_condition_b=True)
    orc = O.Oracle(prob)
    traj = orc.simulate(prob.truth)
    # condition 1: (0,1,2) -> (2,0,2) -> (2,1,2), fixed thereafter (golden header)
    assert traj[1, 1].tolist() == [2, 0, 2]
    for t in range(2, 7):
        assert traj[1, t].tolist() == [2, 1, 2]
    for label, p, nv, want in golden_rows("example_b_fitness.txt"):
        x = prob.truth.copy()
        if int(p) >= 0:
            x[int(p)] = int(nv)
        assert orc.fitness(x) == int(want), label
    # the w[e0] candidate: cond 0 runs (2,0,2),(2,1,0),(2,2,1),(2,1,1),(2,1,1),(2,1,1)
    x = prob.truth.copy(); x[0] = 0
    got = orc.simulate(x)[0, 1:].tolist()
    assert got == [[2, 0, 2], [2, 1, 0], [2, 2, 1], [2, 1, 1], [2, 1, 1], [2, 1, 1]]
    # the theta[1] candidate: cond 0 runs (2,0,2),(2,0,0),(2,1,0),(1,1,1),(2,0,1),(2,1,0); cond 1 sticks
    x = prob.truth.copy(); x[7] = 5
    tr = orc.simulate(x)
    assert tr[0, 1:].tolist() == [[2, 0, 2], [2, 0, 0], [2, 1, 0], [1, 1, 1], [2, 0, 1], [2, 1, 0]]
    assert all(tr[1, t].tolist() == [2, 0, 2] for t in range(1, 7))


# ------------------------------------------------------------------ Pin 3: mapping arithmetic
def test_mapping_arithmetic():
    cur_w = np.zeros(9, dtype=np.int8)                       # P=9: 6 weights (all 0) + 3 pair indices (0)
    for row in golden_rows("mapping.txt"):
        kind, x, want = row[0], int(row[1], 0), int(row[2])
        if kind == "index":
            p, _ = O.propose(x, 0, 9, 6, 6, cur_w)
            assert p == want and O.mulhi(x, 9) == want
        elif kind == "woff":
            # weight 0 (code 1): new code = (1 + off) % 3 -> off=1 gives +1, off=2 gives -1
            p, nv = O.propose(0, x, 9, 6, 6, cur_w)
            assert p == 0 and nv == ((1 + want) % 3) - 1
        elif kind == "poff":
            p, nv = O.propose(0xFFFFFFFF, x, 9, 6, 6, cur_w)
            assert p == 8 and nv == want % 6
        elif kind == "accept":
            row_t1 = O.geometric_table(1.0, 1.0, 1, 64)[0]
            assert row_t1[0] == 1580030168
            assert O.accept(1, x, row_t1) == bool(want)
    # proposals are never a no-op and stay in range, for every old value
    for old in (-1, 0, 1):
        cur = np.full(9, old, dtype=np.int8); cur[6:] = 0
        seen = set()
        for x1 in (0, 0x7FFFFFFF, 0x80000000, 0xFFFFFFFF):
            _, nv = O.propose(0, x1, 9, 6, 6, cur)
            assert nv != old and nv in (-1, 0, 1)
            seen.add(nv)
        assert len(seen) == 2                                 # both other values reachable
    for old in range(6):
        cur = np.zeros(9, dtype=np.int8); cur[8] = old
        seen = set()
        for x1 in (0x00000000, 0x33333334, 0x66666667, 0x9999999A, 0xCCCCCCCD):
            _, nv = O.propose(0xFFFFFFFF, x1, 9, 6, 6, cur)
            assert nv != old and 0 <= nv < 6
            seen.add(nv)
        assert len(seen) == 5
    # d <= 0 always accepted, d > D always rejected
    row = np.full(64, 0, dtype=np.uint32)
    assert O.accept(0, 0xFFFFFFFF, row) and O.accept(-5, 0xFFFFFFFF, row)
    assert not O.accept(65, 0, np.full(64, 0xFFFFFFFF, dtype=np.uint32))


# ------------------------------------------------------------------ Pin 4: table closed form
def test_accept_table_closed_form():
    for T, d, want in golden_rows("accept_table.txt"):
        T, d, want = float(T), int(d), int(want)
        tab = O.geometric_table(T, T, 1, 64)
        assert int(tab[0, d - 1]) == want
        assert int(PB.geometric_table(T, T, 1, 64)[0, d - 1]) == want
    tab = O.geometric_table(PB.T0, PB.T_END, PB.N_LEVELS, PB.DMAX)
    assert np.array_equal(tab, PB.geometric_table(PB.T0, PB.T_END, PB.N_LEVELS, PB.DMAX))
    assert (np.diff(tab.astype(np.int64), axis=1) <= 0).all()     # non-increasing in d
    assert (np.diff(tab.astype(np.int64), axis=0) <= 0).all()     # non-increasing in level
    assert int(tab[0, 0]) == 3344923893 and int(tab[-1, 0]) == 8 and int(tab[-1, 1]) == 0


# ------------------------------------------------------------------ Pin 5: all weights zero
@pytest.mark.parametrize("name", ["tiny", "hpg", "mtb"])
def test_all_zero_weights_closed_form(problems_cache, name):
    prob = problems_cache(name)
    rng = np.random.default_rng(5)
    x = np.zeros(prob.n_params, dtype=np.int8)
    x[prob.n_edges:] = rng.integers(0, 6, prob.n_nodes)
    fixed = np.array([2, 1, 1, 1, 1, 0], dtype=np.uint8)[x[prob.n_edges:]]
    traj = O.Oracle(prob).simulate(x)
    want = 0
    for k in range(prob.n_cond):
        expect = np.where(prob.clamp[k] == 1, prob.init_state[k], fixed)
        for t in range(1, prob.n_steps + 1):
            assert np.array_equal(traj[k, t], expect)
        for j in range(prob.n_obs):
            o = prob.obs[k, j]
            want += int(((o != 255) & (o != expect)).sum())
    assert O.Oracle(prob).fitness(x) == want


# ------------------------------------------------------------------ dense library-matmul special case
def _dense_fitness(prob, X):
    """Fitness through a dense weight matrix and numpy matmul (library routine as the step)."""
    X = np.atleast_2d(X)
    n, N, E = X.shape[0], prob.n_nodes, prob.n_edges
    W = np.zeros((n, N, N), dtype=np.int32)
    W[:, prob.edge_dst, prob.edge_src] = X[:, :E]
    lo = prob.th_lo.astype(np.int32)[X[:, E:]]
    hi = prob.th_hi.astype(np.int32)[X[:, E:]]
    fit = np.zeros(n, dtype=np.int64)
    for k in range(prob.n_cond):
        s = np.broadcast_to(prob.init_state[k].astype(np.int32), (n, N)).copy()
        for t in range(1, prob.n_steps + 1):
            tot = np.matmul(W, s[:, :, None])[:, :, 0]
            s2 = np.where(tot < lo, 0, np.where(tot > hi, 2, 1))
            s = np.where(prob.clamp[k][None, :] == 1, prob.init_state[k][None, :].astype(np.int32), s2)
            for j, tj in enumerate(prob.obs_times):
                if tj == t:
                    o = prob.obs[k, j].astype(np.int32)
                    fit += ((o[None, :] != 255) & (o[None, :] != s)).sum(axis=1)
    return fit


@pytest.mark.parametrize("name", ["tiny", "hpg", "mtb"])
def test_fitness_equals_dense_matmul(problems_cache, name):
    prob = problems_cache(name)
    X = PB.random_params(prob, 24, seed=11)
    got = O.Oracle(prob).fitness_batch(X)
    assert np.array_equal(got.astype(np.int64), _dense_fitness(prob, X))


# ------------------------------------------------------------------ Pin 6: invariants
@pytest.mark.parametrize("name", ["tiny", "hpg", "mtb", "large"])
def test_ground_truth_invariants(problems_cache, name):
    prob = problems_cache(name)
    clean = copy.copy(prob); clean.obs = prob.obs_clean
    assert O.Oracle(clean).fitness(prob.truth) == 0              # (i) y = 0 on self-generated data
    assert O.Oracle(prob).fitness(prob.truth) == prob.n_flipped  # (ii)
    assert prob.n_flipped == {"tiny": 2, "hpg": 16, "mtb": 179, "large": 3558}[name]
    traj = O.Oracle(prob).simulate(prob.truth)
    assert traj.max() <= 2                                       # (iii)
    X = PB.random_params(prob, 4, seed=3)
    f = O.Oracle(prob).fitness_batch(X)
    assert (f <= prob.n_scored).all()
    assert prob.alg_ops_per_step == {"tiny": 1088, "hpg": 13568, "mtb": 310784, "large": 6727168}[name]


@pytest.mark.parametrize("name", ["tiny", "hpg", "mtb"])
def test_relabelling_and_edge_order_invariance(problems_cache, name):
    prob = problems_cache(name)
    rng = np.random.default_rng(9)
    X = PB.random_params(prob, 6, seed=4)
    base = O.Oracle(prob).fitness_batch(X)
    N, E = prob.n_nodes, prob.n_edges
    perm = rng.permutation(N)                      # node i -> perm[i]
    eperm = rng.permutation(E)                     # new edge e' = old edge eperm[e']
    q = copy.copy(prob)
    q.edge_src = perm[prob.edge_src][eperm].astype(np.int32)
    q.edge_dst = perm[prob.edge_dst][eperm].astype(np.int32)
    inv = np.argsort(perm)
    q.init_state = prob.init_state[:, inv]
    q.clamp = prob.clamp[:, inv]
    q.obs = prob.obs[:, :, inv]
    Xq = np.concatenate([X[:, :E][:, eperm], X[:, E:][:, inv]], axis=1)
    assert np.array_equal(O.Oracle(q).fitness_batch(Xq), base)   # (iv)


def test_weight_into_always_clamped_node_is_inert(problems_cache):
    prob = copy.copy(problems_cache("hpg"))
    node = int(prob.edge_dst[0])
    prob.clamp = prob.clamp.copy(); prob.clamp[:, node] = 1
    orc = O.Oracle(prob)
    X = PB.random_params(prob, 5, seed=8)
    for x in X:
        f0 = orc.fitness(x)
        for e in np.nonzero(prob.edge_dst == node)[0]:
            for w in (-1, 0, 1):
                y = x.copy(); y[e] = w
                assert orc.fitness(y) == f0                        # (v)
        for q in range(6):                                        # its threshold is inert too
            y = x.copy(); y[prob.n_edges + node] = q
            assert orc.fitness(y) == f0


@pytest.mark.parametrize("name", ["tiny", "hpg"])
def test_sa_run_invariants(problems_cache, name):
    prob = problems_cache(name)
    orc = O.Oracle(prob)
    sched = PB.default_schedule(name, total_steps=2000)
    for chain in (0, 3):
        full = orc.run_chain(sched, chain, 600)
        tr = O.unpack_trace(full["trace"])
        # replay the trace: (vi) d_best non-increasing, d_best <= d_cur, fitness consistent
        x, f0 = orc.init_chain(sched.seed, chain)
        assert f0 == full["init_fit"]
        fc = fb = f0
        best = x.copy()
        for g in range(600):
            p, code = int(tr["param"][g]), int(tr["code"][g])
            nv = code - 1 if p < prob.n_edges else code
            assert nv != x[p]
            if tr["accepted"][g]:
                x[p] = nv
                fc = int(tr["delta_cand"][g])
                if tr["new_best"][g]:
                    assert fc < fb
                    fb, best = fc, x.copy()
                else:
                    assert fc >= fb
            else:
                assert not tr["new_best"][g]
            assert fb <= fc
            if g % 97 == 0:
                assert orc.fitness(x) == fc and orc.fitness(best) == fb
        assert np.array_equal(x, full["cur"]) and np.array_equal(best, full["best"])
        assert fc == full["fit_cur"] and fb == full["fit_best"]
        assert orc.fitness(full["cur"]) == full["fit_cur"] and orc.fitness(full["best"]) == full["fit_best"]
        # (vii) run(a); run(b) == run(a+b)
        a = orc.run_chain(sched, chain, 250)
        b = orc.run_chain(sched, chain, 350, g0=250, state=(a["cur"], a["best"], a["fit_cur"], a["fit_best"]))
        assert np.array_equal(b["cur"], full["cur"]) and np.array_equal(b["best"], full["best"])
        assert np.array_equal(np.concatenate([a["trace"], b["trace"]]), full["trace"])
    # chains differ from one another
    assert not np.array_equal(orc.run_chain(sched, 0, 50)["trace"], orc.run_chain(sched, 1, 50)["trace"])


def test_extreme_tables(problems_cache):
    prob = problems_cache("hpg")
    orc = O.Oracle(prob)
    greedy = PB.make_schedule(4, 400)
    greedy.accept = np.zeros_like(greedy.accept)
    r = orc.run_chain(greedy, 1, 400)
    tr = O.unpack_trace(r["trace"])
    fc = r["init_fit"]
    for g in range(400):                                          # (viii) all-zero table: greedy
        if tr["accepted"][g]:
            assert int(tr["delta_cand"][g]) <= fc
            fc = int(tr["delta_cand"][g])
        else:
            assert int(tr["delta_cand"][g]) > fc
    hot = PB.make_schedule(4, 400, dmax=prob.n_scored)
    hot.accept = np.full((hot.n_levels, prob.n_scored), 0xFFFFFFFF, dtype=np.uint32)
    r = orc.run_chain(hot, 1, 400)
    tr = O.unpack_trace(r["trace"])
    # x2 == 0xFFFFFFFF would still be rejected (strict <); with 400 draws that does not occur
    assert tr["accepted"].all()


# ------------------------------------------------------------------ Pin 7: brute force
def test_brute_force_4_nodes_6_edges():
    prob = brute_force_problem(O.simulate_fn)
    assert prob.n_nodes == 4 and prob.n_edges == 6 and prob.n_flipped == 0
    X = all_settings(6, 4, 6)
    assert X.shape[0] == 944784
    orc = O.Oracle(prob)
    fit = orc.fitness_batch(X, threads=min(8, os.cpu_count() or 1))
    assert fit.min() == 0                                         # noise-free data: y = 0 is reachable ...
    row = 0
    for e in range(6):
        row += (int(prob.truth[e]) + 1) * 3 ** e
    for i in range(4):
        row += int(prob.truth[6 + i]) * 3 ** 6 * 6 ** i
    assert np.array_equal(X[row], prob.truth) and fit[row] == 0   # ... and attained by the ground truth
    assert fit.max() <= prob.n_scored
    # the whole array again through the dense library-matmul route
    dense = np.concatenate([_dense_fitness(prob, X[a:a + 65536]) for a in range(0, X.shape[0], 65536)])
    assert np.array_equal(fit.astype(np.int64), dense)


# ------------------------------------------------------------------ Pin 8: Philox vs ATen's engine
def test_philox_matches_aten_engine():
    cases = [(42, 0, 0, 0), (42, 7, 0, 123456), (0xDEADBEEFCAFEF00D, 4095, 1, 0x1_0000_0005),
             (1, 0xFFFFFFFF, 1, 0xFFFFFFFF), (0, 0, 0, 1), (42, 65535, 0, 19999)]
    blocks = aten_philox_blocks([(seed, chain | (domain << 32), g) for seed, chain, domain, g in cases])
    for (seed, chain, domain, g), want in zip(cases, blocks):
        got = O.philox4x32_10([g & 0xFFFFFFFF, g >> 32, chain, domain], [seed & 0xFFFFFFFF, seed >> 32])
        assert got == want, (seed, chain, domain, g)
    # counters differing in one word give unrelated blocks
    a = O.philox4x32_10([0, 0, 0, 0], [42, 0])
    for ctr in ([1, 0, 0, 0], [0, 1, 0, 0], [0, 0, 1, 0], [0, 0, 0, 1]):
        assert O.philox4x32_10(ctr, [42, 0]) != a


# ------------------------------------------------------------------ the wiring of one chain step
def _level_gated_table(n_levels, dmax):
    """Row l accepts a worse move with probability 1/2 iff d <= l (threshold 2^31 up to d = l, 0
    beyond): rows differ strongly by level, so a level index that is off by one or does not saturate
    changes decisions, and the decision depends on the value of x2, so another word in its place does too."""
    tab = np.zeros((n_levels, dmax), dtype=np.uint32)
    for l in range(n_levels):
        tab[l, :min(l, dmax)] = 0x80000000
    return tab


@pytest.mark.parametrize("name,chain,g0", [("tiny", 3, 0), ("hpg", 5, 0), ("tiny", 2, (1 << 32) - 60)])
def test_chain_step_wiring_recomputed_outside_the_oracle(problems_cache, name, chain, g0):
    """SURVEY.md §8(c)-3 / PAPER.md Table 1 :130-149, recomputed step by step OUTSIDE orc_run_chain
    from independently pinned pieces: the random block from ATen's Philox engine (seed, subsequence =
    chain | 0 << 32, offset = g), the index and the new value by integer arithmetic written here,
    delta_cand from Oracle.fitness (Pins 1, 2, 5, 7), level = min(g // spl, L-1), accept iff d <= 0 or
    (d <= D and x2 < table[level][d-1]).  Fails if orc_run_chain swaps counter words, uses domain 1,
    feeds x1 / x3 to the accept test, is off by one in the level or does not saturate it."""
    prob = problems_cache(name)
    orc = O.Oracle(prob)
    E, NP, n_pairs = prob.n_edges, prob.n_params, prob.n_pairs
    L, spl, D, n = 8, 20, 6, 230                                      # L * spl = 160 < 230: 70 saturated steps
    sched = PB.make_schedule(8, L * spl, n_levels=L, dmax=D)
    sched.accept = _level_gated_table(L, D)
    assert sched.steps_per_level == spl
    cur, f0 = orc.init_chain(sched.seed, chain)
    state = None
    if g0:                                                           # start far along: g no longer fits 32 bits midway
        state = (cur, cur.copy(), f0, f0)
    run = orc.run_chain(sched, chain, n, g0=g0, state=state)
    tr = O.unpack_trace(run["trace"])
    blocks = aten_philox_blocks([(sched.seed, chain, g0 + it) for it in range(n)])
    x = cur.copy()
    best, fc, fb = x.copy(), f0, f0
    seen_levels, gated = set(), 0
    for it in range(n):
        g = g0 + it
        x0, x1, x2, _x3 = blocks[it]
        p = (x0 * NP) >> 32
        if p < E:
            nv = (int(x[p]) + 1 + 1 + ((x1 * 2) >> 32)) % 3 - 1
        else:
            nv = (int(x[p]) + 1 + ((x1 * (n_pairs - 1)) >> 32)) % n_pairs
        cand = x.copy()
        cand[p] = nv
        fcand = orc.fitness(cand)
        d = fcand - fc
        level = min(g // spl, L - 1)
        acc = d <= 0 or (d <= D and x2 < int(sched.accept[level][d - 1]))
        if 0 < d <= D:
            gated += 1
            seen_levels.add(level)
        new_best = acc and fcand < fb
        assert int(tr["param"][it]) == p, (it, "parameter index")
        assert int(tr["code"][it]) == (nv + 1 if p < E else nv), (it, "new value")
        assert int(tr["delta_cand"][it]) == fcand, (it, "candidate fitness")
        assert bool(tr["accepted"][it]) == acc, (it, "accept decision", d, level)
        assert bool(tr["new_best"][it]) == new_best, (it, "new best")
        if acc:
            x, fc = cand, fcand
            if new_best:
                best, fb = cand.copy(), fcand
    assert np.array_equal(x, run["cur"]) and np.array_equal(best, run["best"])
    assert (fc, fb) == (run["fit_cur"], run["fit_best"])
    if g0 == 0:
        assert gated >= 20 and len(seen_levels) >= 4                  # the level-dependent branch was exercised
    else:
        assert g0 + n > (1 << 32)                                     # the high counter word was exercised


def test_accept_boundaries():
    """d == D is still looked up (last column), d == D + 1 is rejected whatever the row holds."""
    D = 6
    ones = np.full(D, 0xFFFFFFFF, dtype=np.uint32)
    assert O.accept(D, 0, ones) is True and O.accept(D, 0xFFFFFFFE, ones) is True
    assert O.accept(D, 0xFFFFFFFF, ones) is False                    # strict <
    assert O.accept(D + 1, 0, ones) is False
    last_only = np.zeros(D, dtype=np.uint32); last_only[D - 1] = 7
    assert O.accept(D, 6, last_only) is True and O.accept(D, 7, last_only) is False
    assert O.accept(D - 1, 0, last_only) is False                    # column d-1, not d


def test_chain_init_uses_domain_1(problems_cache):
    prob = problems_cache("hpg")
    orc = O.Oracle(prob)
    x, _ = orc.init_chain(42, 5)
    y = O.philox4x32_10([0, 0, 5, 1], [42, 0])
    assert [int(v) for v in x[:4]] == [O.mulhi(v, 3) - 1 for v in y]
    q = (prob.n_edges + 3) // 4            # first block that holds only threshold indices or the boundary
    y = O.philox4x32_10([q, 0, 5, 1], [42, 0])
    for m in range(4):
        p = 4 * q + m
        if p < prob.n_params:
            want = O.mulhi(y[m], 3) - 1 if p < prob.n_edges else O.mulhi(y[m], 6)
            assert int(x[p]) == want
    assert set(np.unique(x[:prob.n_edges])) <= {-1, 0, 1} and x[prob.n_edges:].max() <= 5 and x[prob.n_edges:].min() >= 0
