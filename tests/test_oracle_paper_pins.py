"""Pins for the paper-model CPU oracle (oracle/sa_oracle_paper.cpp).
None of these retypes the oracle's own formulas: hand-worked values (tests/golden), counts the paper
prints, special cases that reduce to the pinned synchronous oracle, brute force on a tiny network, and
the chain step recomputed outside the oracle from ATen's Philox engine."""
import itertools

import numpy as np
import pytest

from oracle import oracle as O
from oracle import oracle_paper as OP
from paper_2506_19866_b200 import problems as PB
from helpers import aten_philox_blocks, golden_rows


def example_c(ref=None, fast=(0, 0, 0), T=8):
    """The 3-node / 5-edge network of tests/golden/example_c_priority.txt."""
    src = np.array([0, 1, 2, 1, 0], dtype=np.int32)
    dst = np.array([1, 2, 0, 0, 2], dtype=np.int32)
    #                 w              p                 t              u        m        d
    truth = np.array([1, 1, 2, 1, 1, 1, -1, 1, -1, 1, 1, 1, 1, 2, 2, 3, 3, 2, 0, 0, 2, 1, 2, 1], dtype=np.int8)
    init = np.array([[0, 2, 2]], dtype=np.uint8)
    if ref is None:
        ref = np.full((1, T + 1, 3), 255, dtype=np.uint8)
    return PB.PaperProblem(name="example_c", seed=0, n_nodes=3, n_edges=5, edge_src=src, edge_dst=dst,
                           fast=np.array(fast, dtype=np.uint8), n_cond=1, n_steps=T, init_state=init, ref=ref, truth=truth)


@pytest.fixture(scope="module")
def paper_problems():
    cache = {}

    def get(name):
        if name not in cache:
            cache[name] = PB.make_paper_problem(name, OP.simulate_fn)
        return cache[name]
    return get


# ------------------------------------------------------------------ hand-worked examples
def test_example_c_priority_update():
    prob = example_c()
    traj = OP.PaperOracle(prob).simulate(prob.truth)[0]
    rows = golden_rows("example_c_priority.txt")
    assert len(rows) == 9
    for r in rows:
        t, want = int(r[0]), [int(v) for v in r[1:]]
        assert traj[t].tolist() == want, f"t={t}"


def test_example_e_memory_rules():
    src = np.array([0, 1, 2], dtype=np.int32)
    dst = np.array([1, 2, 0], dtype=np.int32)
    #             w        p         t        u        m        d
    x = np.array([1, 1, 1, 1, -1, 1, 1, 1, 1, 1, 3, 1, 0, 1, 0, 1, 1, 2], dtype=np.int8)
    prob = PB.PaperProblem(name="example_e", seed=0, n_nodes=3, n_edges=3, edge_src=src, edge_dst=dst,
                           fast=np.zeros(3, dtype=np.uint8), n_cond=1, n_steps=7,
                           init_state=np.array([[2, 0, 2]], dtype=np.uint8), ref=np.full((1, 8, 3), 255, dtype=np.uint8))
    traj = OP.PaperOracle(prob).simulate(x)[0]
    rows = golden_rows("example_e_memory.txt")
    assert len(rows) == 8
    for r in rows:
        assert traj[int(r[0])].tolist() == [int(v) for v in r[1:]], f"t={r[0]}"


def test_example_d_objective():
    rows = golden_rows("example_d_objective.txt")
    ref = np.full((1, 9, 3), 255, dtype=np.uint8)
    want = {}
    for r in rows:
        if r[0] == "R":
            ref[0, :, int(r[1])] = [int(v) for v in r[2:]]
        else:
            want[r[0]] = int(r[1])
    prob = example_c(ref)
    orc = OP.PaperOracle(prob)
    assert orc.objective(prob.truth) == want["y"] == 15
    s = orc.simulate(prob.truth)[0].astype(int)
    m = ref[0] != 255
    assert int(np.abs(s - ref[0].astype(int))[m].sum()) == want["manhattan"] == 6
    # R = S on the measured nodes: y = 0
    same = np.full((1, 9, 3), 255, dtype=np.uint8)
    same[0, :, 0], same[0, :, 2] = s[:, 0], s[:, 2]
    assert OP.PaperOracle(example_c(same)).objective(prob.truth) == 0
    # measuring node 1 as well, with a reference equal to what it does, adds nothing
    more = ref.copy(); more[0, :, 1] = s[:, 1]
    assert OP.PaperOracle(example_c(more)).objective(prob.truth) == 15
    # a constant reference has G = 0 everywhere: y is the plain Manhattan distance
    flat = np.full((1, 9, 3), 255, dtype=np.uint8); flat[0, :, 0] = 1
    assert OP.PaperOracle(example_c(flat)).objective(prob.truth) == int(np.abs(s[:, 0] - 1).sum())


# ------------------------------------------------------------------ what the paper prints
def test_parameter_counts_and_level_count(paper_problems):
    """102 = 3*25 + 3*9 and 723 = 3*178 + 3*63; :115: T 1000 -> 0.001 at rho 0.99."""
    assert paper_problems("paper_hpg").n_params == 102
    assert paper_problems("paper_mtb").n_params == 723
    assert PB.paper_levels() == 1375
    p = paper_problems("paper_mtb")
    assert (p.n_nodes, p.n_edges, len(p.measured_nodes), int(p.fast.sum()), p.n_steps + 1) == (63, 178, 35, 21, 20)
    h = paper_problems("paper_hpg")
    assert (h.n_nodes, h.n_edges, len(h.measured_nodes), int(h.fast.sum()), h.n_steps + 1) == (9, 25, 5, 3, 20)


@pytest.mark.parametrize("name", ["paper_tiny", "paper_hpg", "paper_mtb"])
def test_ground_truth_and_trajectory_invariants(paper_problems, name):
    import copy
    prob = paper_problems(name)
    orc = OP.PaperOracle(prob)
    clean = copy.copy(prob); clean.ref = prob.ref_clean
    assert OP.PaperOracle(clean).objective(prob.truth) == 0            # y = 0 on self-generated data (:245, :263)
    assert orc.valid(prob.truth)
    if prob.n_flipped == 0:
        assert orc.objective(prob.truth) == 0
    else:
        assert 0 < orc.objective(prob.truth) <= 6 * 3 * prob.n_flipped    # a flip touches its own and the next row's weight
    E, N = prob.n_edges, prob.n_nodes
    for x in PB.random_paper_params(prob, 6, seed=2):
        traj = orc.simulate(x).astype(int)
        assert traj.max() <= 2 and np.array_equal(traj[:, 0], prob.init_state)
        step = np.abs(np.diff(traj, axis=1))                           # [K][T][N]
        d = x[3 * E + 2 * N:].astype(int)
        m = x[3 * E + N:3 * E + 2 * N].astype(int)
        assert (step <= d[None, None, :]).all()                        # at most d_i levels per time step (:80)
        for i in range(N):
            assert (step[:, :m[i], i] == 0).all()                      # told m_i times first (:79): nothing moves before t = m_i + 1
        assert orc.objective(x) <= prob.max_objective


# ------------------------------------------------------------------ where the two models coincide
def _as_sync_problem(prob):
    """The same structure as a config-model problem whose single threshold pair (1, 1) makes the
    synchronous rule s' = 0 if sum < 1, 2 if sum > 1, else 1 equal to clip(sum, 0, 2)."""
    N = prob.n_nodes
    return PB.Problem(name="sync", seed=0, n_nodes=N, n_edges=prob.n_edges, edge_src=prob.edge_src, edge_dst=prob.edge_dst,
                      th_lo=np.array([1], dtype=np.int8), th_hi=np.array([1], dtype=np.int8), n_cond=prob.n_cond, n_steps=1,
                      obs_times=np.array([1], dtype=np.int32), init_state=prob.init_state,
                      clamp=np.zeros_like(prob.init_state), obs=np.full((prob.n_cond, 1, N), 255, dtype=np.uint8))


@pytest.mark.parametrize("name", ["paper_tiny", "paper_hpg", "paper_mtb"])
def test_first_transition_reduces_to_the_synchronous_rule(paper_problems, name):
    """With w in {0,1}, t = 1, every u equal, m = 0 and d = 2, all nodes that differ from their image
    share one priority at t = 1 and jump straight to it: s(1) = clip(SUM p*w*s_j, 0, 2) — the pinned
    synchronous oracle with signed weights p*w and the pair (1, 1).  With d = 1 instead they move one
    level toward that value."""
    prob = paper_problems(name)
    E, N = prob.n_edges, prob.n_nodes
    rng = np.random.default_rng(7)
    sync = O.Oracle(_as_sync_problem(prob))
    porc = OP.PaperOracle(prob)
    lay = prob.layout()
    for trial in range(12):
        x = np.zeros(prob.n_params, dtype=np.int8)
        x[lay["w"]:lay["w"] + E] = rng.integers(0, 2, E)
        x[lay["p"]:lay["p"] + E] = rng.integers(-1, 2, E)
        x[lay["t"]:lay["t"] + E] = 1
        x[lay["u"]:lay["u"] + N] = 5
        x[lay["m"]:lay["m"] + N] = 0
        x[lay["d"]:lay["d"] + N] = 2
        signed = (x[lay["w"]:lay["w"] + E] * x[lay["p"]:lay["p"] + E]).astype(np.int8)
        want = sync.simulate(np.concatenate([signed, np.zeros(N, dtype=np.int8)]))[:, 1]      # [K][N]
        got = porc.simulate(x)[:, 1]
        assert np.array_equal(got, want)
        x[lay["d"]:lay["d"] + N] = 1
        one = porc.simulate(x)[:, 1].astype(int)
        s0 = prob.init_state.astype(int)
        assert np.array_equal(one, s0 + np.sign(want.astype(int) - s0))


def test_single_edge_image_for_every_state_weight_polarity_threshold():
    """One live edge 0 -> 1 (the edge back has weight 0, so node 0's image is 0): node 1 has the higher
    speed and d = 2, so whenever its image differs from its state it alone moves, straight to
    clip((s_0 // t) * w * p, 0, 2) (t is the minimum level of s_j for the interaction
    to be active, floor division); otherwise node 0 decays to its image 0."""
    src, dst = np.array([0, 1], dtype=np.int32), np.array([1, 0], dtype=np.int32)
    floor_div = {(0, 1): 0, (1, 1): 1, (2, 1): 2, (0, 2): 0, (1, 2): 0, (2, 2): 1}      # s // t written out
    for s0, s1, w, p, t in itertools.product((0, 1, 2), (0, 1, 2), (0, 1, 2), (-1, 0, 1), (1, 2)):
        prob = PB.PaperProblem(name="edge", seed=0, n_nodes=2, n_edges=2, edge_src=src, edge_dst=dst,
                               fast=np.zeros(2, dtype=np.uint8), n_cond=1, n_steps=1,
                               init_state=np.array([[s0, s1]], dtype=np.uint8), ref=np.full((1, 2, 2), 255, dtype=np.uint8))
        x = np.array([w, 0, p, 0, t, 1, 1, 6, 0, 0, 2, 2], dtype=np.int8)          # u = (1, 6), m = 0, d = 2
        image = floor_div[(s0, t)] * w * p
        target = min(2, max(0, image))
        got = OP.PaperOracle(prob).simulate(x)[0, 1].tolist()
        assert got == ([s0, target] if target != s1 else [0, s1]), (s0, s1, w, p, t)


# ------------------------------------------------------------------ value ranges and GetCandidate mapping
def test_mapping_arithmetic():
    prob = example_c(fast=(0, 1, 0))
    orc = OP.PaperOracle(prob)
    assert [orc.domain(q) for q in (0, 5, 10, 15, 16, 18, 21)] == [[0, 1, 2], [-1, 0, 1], [1, 2], [1, 2, 3, 4, 5, 6],
                                                                    [10, 11, 12], [0, 1, 2], [1, 2]]
    base = prob.truth.copy(); base[16] = 10
    for row in golden_rows("paper_mapping.txt"):
        if row[0] == "index":
            q, _, moved = orc.propose(int(row[1], 0), 0, base)
            assert q == int(row[2]) and moved
        elif row[0] == "value":
            q, old, x1, want = int(row[1]), int(row[2]), int(row[3], 0), int(row[4])
            cur = base.copy(); cur[q] = old
            x0 = ((q << 32) + 23) // 24 + 1                     # some x0 with floor(x0 * 24 / 2^32) = q
            got_q, nv, moved = orc.propose(x0, x1, cur)
            assert (got_q, nv, moved) == (q, want, True), row
        elif row[0] == "init":
            q, y, want = int(row[1]), int(row[2], 0), int(row[3])
            dom = orc.domain(q)
            assert dom[(y * len(dom)) >> 32] == want, row
    # never a no-op, every other value reachable, for every parameter and old value
    for q in range(24):
        dom = orc.domain(q)
        for old in dom:
            cur = base.copy(); cur[q] = old
            seen = set()
            for k in range(len(dom) - 1):
                x1 = min(0xFFFFFFFF, ((k << 32) + len(dom) - 2) // (len(dom) - 1) + 1) if k else 0
                seen.add(orc.propose(((q << 32) + 23) // 24 + 1, x1, cur)[1])
            assert seen == set(dom) - {old}


def test_initial_vector_follows_the_philox_blocks(paper_problems):
    """Unconstrained: parameter 4b+j = domain[mulhi(y_j, size)] of block Philox(ctr = (b, 0, chain, 1));
    constrained: the repair pass recomputed here from ATen's blocks of domain 2."""
    prob = paper_problems("paper_hpg")
    orc = OP.PaperOracle(prob)
    E, N, NP = prob.n_edges, prob.n_nodes, prob.n_params
    seed, chain = 42, 9
    nb = (NP + 3) // 4
    blocks = aten_philox_blocks([(seed, chain | (1 << 32), b) for b in range(nb)])
    x, _ = orc.init_chain(seed, chain, constrained=False)
    want = np.zeros(NP, dtype=np.int8)
    for q in range(NP):
        dom = PB.paper_domain(prob, q)
        want[q] = dom[(blocks[q // 4][q % 4] * len(dom)) >> 32]
    assert np.array_equal(x, want)
    repaired_any = False
    for chain in range(40):
        blocks = aten_philox_blocks([(seed, chain | (1 << 32), b) for b in range(nb)])
        rep = aten_philox_blocks([(seed, chain | (2 << 32), i) for i in range(N)])
        v = np.zeros(NP, dtype=np.int8)
        for q in range(NP):
            dom = PB.paper_domain(prob, q)
            v[q] = dom[(blocks[q // 4][q % 4] * len(dom)) >> 32]
        ins = [[e for e in range(E) if prob.edge_dst[e] == i] for i in range(N)]
        outs = [[e for e in range(E) if prob.edge_src[e] == i] for i in range(N)]
        for i in range(N):
            if not any(v[E + e] == 1 and v[e] != 0 for e in ins[i]):
                e = ins[i][(rep[i][0] * len(ins[i])) >> 32]
                v[E + e] = 1
                if v[e] == 0:
                    v[e] = 1 + ((rep[i][1] * 2) >> 32)
                repaired_any = True
        for i in range(N):
            if not any(v[e] != 0 for e in outs[i]):
                e = outs[i][(rep[i][2] * len(outs[i])) >> 32]
                v[e] = 1 + ((rep[i][3] * 2) >> 32)
                repaired_any = True
        got, _ = orc.init_chain(seed, chain, constrained=True)
        assert np.array_equal(got, v), chain
        assert orc.valid(got)
    assert repaired_any


# ------------------------------------------------------------------ constraints
def test_validity_hand_cases():
    """(a) every node keeps an in- and an out-edge of non-zero weight; (b) every node
    has an in-edge with p = +1 and w != 0.  Example C's network: in(0) = {e2, e3}, in(1) = {e0},
    in(2) = {e1, e4}; out(0) = {e0, e4}, out(1) = {e1, e3}, out(2) = {e2}."""
    prob = example_c()
    orc = OP.PaperOracle(prob)

    def vec(w, p):
        x = prob.truth.copy(); x[0:5] = w; x[5:10] = p
        return x
    assert orc.valid(vec([1, 1, 2, 1, 1], [1, -1, 1, -1, 1]))          # Example C itself
    assert not orc.valid(vec([0, 1, 2, 1, 1], [1, -1, 1, -1, 1]))      # node 1 loses its only in-edge (a)
    assert not orc.valid(vec([1, 1, 0, 1, 1], [1, -1, 1, -1, 1]))      # node 2 loses its only out-edge (a)
    assert not orc.valid(vec([1, 1, 2, 1, 1], [0, -1, 1, -1, 1]))      # node 1's only in-edge no longer activates (b)
    assert not orc.valid(vec([1, 1, 2, 1, 1], [1, -1, -1, -1, 1]))     # node 0: both in-edges inhibit (b)
    assert orc.valid(vec([1, 1, 2, 1, 1], [1, -1, -1, 1, 1]))          # ... unless e3 activates
    assert not orc.valid(vec([1, 1, 2, 0, 1], [1, -1, -1, 1, 1]))      # ... with a non-zero weight (b: w != 0)
    assert orc.valid(vec([1, 0, 2, 1, 1], [1, -1, 1, -1, 1]))          # node 2 still has e4 in, node 1 still has e3 out
    assert not orc.valid(vec([1, 0, 2, 0, 1], [1, -1, 1, -1, 1]))      # node 1 has no out-edge left (a)
    # e4 switched off but e1 now activates node 2: every node keeps an active in-edge and an out-edge
    assert orc.valid(vec([1, 1, 2, 1, 0], [1, 1, 1, -1, -1]))


def test_constrained_getcandidate_brute_force():
    """Every (w, p) setting of Example C's network (9^5 = 59 049): from each VALID vector, for each weight
    or polarity parameter, the constrained GetCandidate reaches exactly the valid neighbours (both halves
    of x1), never an invalid one, and reports a null move iff there is none."""
    prob = example_c()
    orc = OP.PaperOracle(prob)
    n_valid = n_null = n_restricted = 0
    for wp in itertools.product(range(9), repeat=5):
        x = prob.truth.copy()
        for e, c in enumerate(wp):
            x[e], x[5 + e] = c % 3, c // 3 - 1
        if not orc.valid(x):
            continue
        n_valid += 1
        for q in range(10):
            dom = (0, 1, 2) if q < 5 else (-1, 0, 1)
            want = set()
            for v in dom:
                if v != x[q]:
                    y = x.copy(); y[q] = v
                    if orc.valid(y):
                        want.add(v)
            x0 = ((q << 32) + 23) // 24 + 1
            got, null = set(), 0
            for x1 in (0, 0x7FFFFFFF, 0x80000000, 0xFFFFFFFF):
                gq, nv, moved = orc.propose(x0, x1, x, constrained=True)
                assert gq == q
                if moved:
                    got.add(nv)
                else:
                    null += 1
                    assert nv == x[q]
            assert got == want, (wp, q)
            assert (null == 4) == (len(want) == 0) and null in (0, 4)
            n_null += null == 4
            n_restricted += len(want) == 1
            # unconstrained proposals ignore validity
            assert {orc.propose(x0, x1, x)[1] for x1 in (0, 0xFFFFFFFF)} == set(dom) - {int(x[q])}
    assert n_valid > 100 and n_null > 0 and n_restricted > 0


@pytest.mark.parametrize("name", ["paper_tiny", "paper_hpg"])
def test_constrained_chain_stays_valid(paper_problems, name):
    prob = paper_problems(name)
    orc = OP.PaperOracle(prob)
    sched = PB.paper_schedule(4, 20, 30, prob.max_objective)
    for chain in range(3):
        run = orc.run_chain(sched, chain, 600, constrained=True)
        tr = OP.unpack_trace(run["trace"])
        x, _ = orc.init_chain(sched.seed, chain, constrained=True)
        assert orc.valid(x)
        for g in range(600):
            q = int(tr["param"][g])
            nv = PB.paper_domain(prob, q)[int(tr["code"][g])]
            if tr["null_move"][g]:
                assert nv == x[q] and tr["accepted"][g]               # d = 0 is accepted (reading 1)
            else:
                assert nv != x[q]
            if tr["accepted"][g]:
                x[q] = nv
                assert orc.valid(x)
        assert np.array_equal(x, run["cur"]) and orc.valid(run["best"])


# ------------------------------------------------------------------ the wiring of one chain step
@pytest.mark.parametrize("name,chain,constrained,g0", [("paper_tiny", 3, False, 0), ("paper_hpg", 5, True, 0),
                                                        ("paper_tiny", 1, True, (1 << 32) - 50)])
def test_chain_step_wiring_recomputed_outside_the_oracle(paper_problems, name, chain, constrained, g0):
    """PAPER.md Table 1 :130-149 around the pinned pieces: random block from ATen's Philox (seed,
    subsequence = chain | 0 << 32, offset = g), GetCandidate from x0 / x1 (pinned above), y from
    PaperOracle.objective (Examples C / D), level = min(g // spl, L-1), accept iff d <= 0 or (d <= D and
    x2 < table[level][d-1])."""
    prob = paper_problems(name)
    orc = OP.PaperOracle(prob)
    L, spl, D, n = 8, 20, 12, 220
    sched = PB.paper_schedule(8, L, spl, D)
    tab = np.zeros((L, D), dtype=np.uint32)
    for l in range(L):
        tab[l, :min(2 * l, D)] = 0x80000000               # row l: worse by at most 2l accepted with probability 1/2
    sched.accept = tab
    cur, f0 = orc.init_chain(sched.seed, chain, constrained)
    state = (cur, cur.copy(), f0, f0) if g0 else None
    run = orc.run_chain(sched, chain, n, g0=g0, state=state, constrained=constrained)
    tr = OP.unpack_trace(run["trace"])
    blocks = aten_philox_blocks([(sched.seed, chain, g0 + it) for it in range(n)])
    x, best, fc, fb = cur.copy(), cur.copy(), f0, f0
    gated = 0
    for it in range(n):
        g = g0 + it
        x0, x1, x2, _ = blocks[it]
        q, nv, moved = orc.propose(x0, x1, x, constrained)
        assert q == (x0 * prob.n_params) >> 32
        cand = x.copy(); cand[q] = nv
        fcand = orc.objective(cand)
        d = fcand - fc
        level = min(g // spl, L - 1)
        acc = d <= 0 or (d <= D and x2 < int(tab[level][d - 1]))
        gated += 0 < d <= D
        new_best = acc and fcand < fb
        assert int(tr["param"][it]) == q and int(tr["code"][it]) == PB.paper_domain(prob, q).index(nv), it
        assert int(tr["delta_cand"][it]) == fcand, it
        assert bool(tr["accepted"][it]) == acc, (it, d, level)
        assert bool(tr["new_best"][it]) == new_best and bool(tr["null_move"][it]) == (not moved), it
        if acc:
            x, fc = cand, fcand
            if new_best:
                best, fb = cand.copy(), fcand
    assert np.array_equal(x, run["cur"]) and np.array_equal(best, run["best"])
    assert (fc, fb) == (run["fit_cur"], run["fit_best"])
    assert gated >= 10 or g0
    # run(a); run(b) == run(a+b); chains differ
    a = orc.run_chain(sched, chain, 90, g0=g0, state=state, constrained=constrained)
    b = orc.run_chain(sched, chain, n - 90, g0=g0 + 90, state=(a["cur"], a["best"], a["fit_cur"], a["fit_best"]),
                      constrained=constrained)
    assert np.array_equal(np.concatenate([a["trace"], b["trace"]]), run["trace"])
    assert np.array_equal(b["cur"], run["cur"]) and np.array_equal(b["best"], run["best"])
    assert not np.array_equal(orc.run_chain(sched, chain + 1, 40, constrained=constrained)["trace"], run["trace"][:40])
