"""Pins for the structural constraints of PAPER.md §2.5.3 in the config-model oracle (orc_valid,
orc_init_chain_c, orc_propose_c, orc_run_chain_c; readings C1-C3): hand cases, brute force over
every weight setting of a 3-node network, the repair pass and the chain step recomputed outside the oracle
from ATen's Philox."""
import itertools

import numpy as np
import pytest

from oracle import oracle as O
from paper_2506_19866_b200 import problems as PB
from helpers import aten_philox_blocks, example_problem


def test_validity_hand_cases():
    """Example B's network: in(0) = {e0, e1}, in(1) = {e2, e3}, in(2) = {e4, e5}; out(0) = {e2, e4},
    out(1) = {e0, e5}, out(2) = {e1, e3}.  (a) non-zero in- and out-edge, (b) an in-edge with w = +1."""
    prob = example_problem(with_condition_b=True)
    orc = O.Oracle(prob)

    def vec(*w):
        x = prob.truth.copy(); x[:6] = w
        return x
    assert orc.valid(vec(-1, +1, +1, -1, -1, +1))          # Example B itself: +1 into 0 (e1), 1 (e2), 2 (e5)
    assert not orc.valid(vec(-1, 0, +1, -1, -1, +1))       # node 0 loses its activator e1 (b)
    assert not orc.valid(vec(-1, -1, +1, -1, -1, +1))      # ... an inhibitor does not count (b)
    assert orc.valid(vec(+1, 0, +1, -1, -1, +1))           # ... e0 can take over; node 2 still has e3 out
    assert not orc.valid(vec(+1, 0, +1, 0, -1, +1))        # node 2 has no out-edge left (a)
    assert not orc.valid(vec(0, +1, +1, -1, -1, 0))        # node 1 has no out-edge left (a)
    assert not orc.valid(vec(-1, +1, 0, 0, -1, +1))        # node 1 has no in-edge left (a), (b)
    assert orc.valid(vec(+1, +1, +1, +1, +1, +1))
    assert not orc.valid(vec(0, 0, 0, 0, 0, 0))


def test_constrained_getcandidate_brute_force():
    """All 3^6 = 729 weight settings of Example B's network: from every VALID vector and for every weight, the
    constrained GetCandidate reaches exactly the valid neighbours (over both halves of x1), reports a null move
    iff there is none, and agrees with the unconstrained rule when both other values are allowed.  Threshold
    proposals are untouched."""
    prob = example_problem(with_condition_b=True)
    orc = O.Oracle(prob)
    n_valid = n_null = n_one = 0
    for ws in itertools.product((-1, 0, 1), repeat=6):
        x = prob.truth.copy(); x[:6] = ws
        if not orc.valid(x):
            continue
        n_valid += 1
        for p in range(6):
            want = set()
            for v in (-1, 0, 1):
                if v != x[p]:
                    y = x.copy(); y[p] = v
                    if orc.valid(y):
                        want.add(v)
            x0 = ((p << 32) + 8) // 9 + 1                    # some x0 with floor(x0 * 9 / 2^32) = p
            got, null = set(), 0
            for x1 in (0, 0x7FFFFFFF, 0x80000000, 0xFFFFFFFF):
                gp, nv, moved = orc.propose_c(x0, x1, x)
                assert gp == p
                if moved:
                    got.add(nv)
                else:
                    null += 1
                    assert nv == x[p]
                if len(want) == 2:
                    assert (gp, nv) == O.propose(x0, x1, 9, 6, 6, x)
            assert got == want and null in (0, 4) and (null == 4) == (not want), (ws, p)
            n_null += null == 4
            n_one += len(want) == 1
        for p in (6, 7, 8):
            for x1 in (0, 0x55555555, 0xFFFFFFFF):
                x0 = ((p << 32) + 8) // 9 + 1
                gp, nv, moved = orc.propose_c(x0, x1, x)
                assert moved and (gp, nv) == O.propose(x0, x1, 9, 6, 6, x)
    assert n_valid > 50 and n_null > 0 and n_one > 0


@pytest.mark.parametrize("name", ["hpg", "mtb"])
def test_repaired_initial_vector_recomputed_from_aten(problems_cache, name):
    """Reading C3: the unconstrained vector, then node i's block Philox(ctr = (i, 0, chain, 2)) picks the in-edge
    that becomes +1 and the out-edge that becomes +-1 — recomputed here from ATen's engine."""
    prob = problems_cache(name)
    orc = O.Oracle(prob)
    E, N = prob.n_edges, prob.n_nodes
    ins = [[e for e in range(E) if prob.edge_dst[e] == i] for i in range(N)]
    outs = [[e for e in range(E) if prob.edge_src[e] == i] for i in range(N)]
    seed, repaired = 42, 0
    for chain in range(25):
        v, _ = orc.init_chain(seed, chain)
        rep = aten_philox_blocks([(seed, chain | (2 << 32), i) for i in range(N)])
        for i in range(N):
            if not any(v[e] == 1 for e in ins[i]):
                v[ins[i][(rep[i][0] * len(ins[i])) >> 32]] = 1
                repaired += 1
        for i in range(N):
            if not any(v[e] != 0 for e in outs[i]):
                v[outs[i][(rep[i][2] * len(outs[i])) >> 32]] = 2 * ((rep[i][3] * 2) >> 32) - 1
                repaired += 1
        got, f = orc.init_chain(seed, chain, constrained=True)
        assert np.array_equal(got, v), chain
        assert orc.valid(got) and f == orc.fitness(got)
    assert repaired > 0


@pytest.mark.parametrize("name,chain,g0", [("hpg", 4, 0), ("hpg", 2, (1 << 32) - 40)])
def test_constrained_chain_step_wiring(problems_cache, name, chain, g0):
    """orc_run_chain_c recomputed outside the oracle: ATen Philox block (seed, chain, g), orc_propose_c (pinned
    above), Oracle.fitness, level = min(g // spl, L-1), accept iff d <= 0 or (d <= D and x2 < table[level][d-1])."""
    prob = problems_cache(name)
    orc = O.Oracle(prob)
    L, spl, D, n = 8, 20, 6, 220
    sched = PB.make_schedule(8, L * spl, n_levels=L, dmax=D)
    tab = np.zeros((L, D), dtype=np.uint32)
    for l in range(L):
        tab[l, :min(l, D)] = 0x80000000
    sched.accept = tab
    cur, f0 = orc.init_chain(sched.seed, chain, constrained=True)
    state = (cur, cur.copy(), f0, f0) if g0 else None
    run = orc.run_chain(sched, chain, n, g0=g0, state=state, constrained=True)
    tr = O.unpack_trace(run["trace"])
    blocks = aten_philox_blocks([(sched.seed, chain, g0 + it) for it in range(n)])
    x, best, fc, fb = cur.copy(), cur.copy(), f0, f0
    nulls = 0
    for it in range(n):
        g = g0 + it
        x0, x1, x2, _ = blocks[it]
        p, nv, moved = orc.propose_c(x0, x1, x)
        cand = x.copy(); cand[p] = nv
        fcand = orc.fitness(cand)
        d = fcand - fc
        level = min(g // spl, L - 1)
        acc = d <= 0 or (d <= D and x2 < int(tab[level][d - 1]))
        new_best = acc and fcand < fb
        nulls += not moved
        assert int(tr["param"][it]) == p and int(tr["code"][it]) == (nv + 1 if p < prob.n_edges else nv), it
        assert int(tr["delta_cand"][it]) == fcand and bool(tr["accepted"][it]) == acc, (it, d, level)
        assert bool(tr["new_best"][it]) == new_best and bool(tr["null_move"][it]) == (not moved), it
        assert moved or (acc and d == 0)                      # a null move is the current vector: d = 0, accepted
        if acc:
            x, fc = cand, fcand
            assert orc.valid(x)
            if new_best:
                best, fb = cand.copy(), fcand
    assert np.array_equal(x, run["cur"]) and np.array_equal(best, run["best"]) and (fc, fb) == (run["fit_cur"], run["fit_best"])
    assert orc.valid(run["best"])
    if g0 == 0:
        assert nulls > 0
    # the unconstrained chain from the same start differs (the lists differ as soon as a value is struck)
    free = orc.run_chain(sched, chain, n, g0=g0, state=(cur, cur.copy(), f0, f0))
    assert not np.array_equal(free["trace"], run["trace"])


def test_constraints_need_a_closed_loop(problems_cache):
    """tiny has nodes without in-edges: no valid vector exists."""
    orc = O.Oracle(problems_cache("tiny"))
    with pytest.raises(ValueError):
        orc.init_chain(42, 0, constrained=True)
