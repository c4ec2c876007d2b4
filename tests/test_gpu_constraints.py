"""GPU parity of the structural constraints (SA_CONSTRAINED, readings C1-C3) in the
config-model kernels against the constrained config-model oracle.  Needs a GPU (-m gpu)."""
import os

import numpy as np
import pytest

from oracle import oracle as O
from paper_2506_19866_b200 import problems as PB
from test_gpu_parity import B, Handle, NCPU          # noqa: F401  (fixture + helpers)
from concurrent.futures import ThreadPoolExecutor

pytestmark = pytest.mark.gpu


class CHandle(Handle):
    def __init__(self, B, prob, sched, flags=None):
        self.B, self.prob, self.sched = B, prob, sched
        self.h = B.sa_create(prob, sched, flags=B.SA_CONSTRAINED if flags is None else flags)


def oracle_chains(orc, sched, chains, n):
    with ThreadPoolExecutor(NCPU) as ex:
        return list(ex.map(lambda c: orc.run_chain(sched, c + sched.chain_id_base, n, constrained=True), chains))


def check(B, hd, orc, chains, n, trace=None):
    refs = oracle_chains(orc, hd.sched, chains, n)
    for row, (c, ref) in enumerate(zip(chains, refs)):
        cur, fc, best, fb = B.sa_get_chain(hd.h, c, hd.prob.n_params)
        if trace is not None:
            bad = np.nonzero(trace[row][:n] != ref["trace"])[0]
            assert bad.size == 0, f"chain {c}: first trace mismatch at step {bad[0]}: gpu {int(trace[row][bad[0]]):#x} " \
                                  f"oracle {int(ref['trace'][bad[0]]):#x}"
        assert (fc, fb) == (ref["fit_cur"], ref["fit_best"]), c
        assert np.array_equal(cur, ref["cur"]) and np.array_equal(best, ref["best"]), c
        assert orc.valid(cur) and orc.valid(best), c


@pytest.mark.parametrize("name,R", [("hpg", 300), ("mtb", 150), ("large", 12)])
def test_every_chain_starts_from_a_valid_vector(B, problems_cache, name, R):
    prob = problems_cache(name)
    orc = O.Oracle(prob)
    sched = PB.default_schedule(name, n_chains=R, total_steps=400)
    sched.chain_id_base = 7
    with CHandle(B, prob, sched) as hd:
        fc, fb = B.sa_get_fitness(hd.h, R)
        for c in range(R):
            x, f = orc.init_chain(sched.seed, c + 7, constrained=True)
            cur, f1, best, f2 = B.sa_get_chain(hd.h, c, prob.n_params)
            assert np.array_equal(cur, x) and np.array_equal(best, x) and f == f1 == f2 == fc[c] == fb[c], c
            assert orc.valid(cur)


CASES = [("hpg", "STATIC", {}), ("mtb", "STATIC", {}), ("hpg", "GENERIC", {}), ("hpg", "GENERIC", {"TSA_KERNEL": "cta"}), ("hpg", "DENSE", {}), ("hpg", "AUTO", {}),
         ("mtb", "GENERIC", {}), ("mtb", "DENSE", {}), ("mtb", "DENSE", {"TSA_DENSE_SP": "0"}), ("mtb", "DENSE", {"TSA_DENSE_W": "2"}),
         ("mtb", "AUTO", {}), ("mtb", "DENSE", {"TSA_DENSE_MOVM": "1"}), ("mtb", "DENSE", {"TSA_DENSE_CPB": "16"}),
         ("hpg", "DENSE", {"TSA_DENSE_SPEC": "3"}), ("mtb", "DENSE", {"TSA_DENSE_SPEC": "2"})]


@pytest.mark.parametrize("name,family,env", CASES, ids=[f"{n}-{f}-{'-'.join(e.values()) or 'default'}" for n, f, e in CASES])
def test_constrained_traces_match_the_oracle(B, problems_cache, name, family, env):
    prob = problems_cache(name)
    orc = O.Oracle(prob)
    sched = PB.default_schedule(name, n_chains=24, total_steps=600)
    chains = list(range(24))
    os.environ.update(env)
    try:
        with CHandle(B, prob, sched) as hd:
            B.sa_select_kernel(hd.h, getattr(B, "SA_KERNEL_" + family))
            B.sa_set_trace(hd.h, chains, 600)
            B.sa_run(hd.h, 170)
            B.sa_run(hd.h, 430)
            info = B.sa_get_info(hd.h)
            if family in ("DENSE", "AUTO"):
                assert info["variant"] == 5
            if family == "STATIC":
                assert info["variant"] == 4
            tr = B.sa_get_trace(hd.h, 24, 600)
            check(B, hd, orc, chains, 600, tr)
            assert (O.unpack_trace(tr)["null_move"]).any()                # the struck-list branch was exercised
    finally:
        for k in env:
            del os.environ[k]


def test_constraints_with_balanced_slots_levels_and_statistics(B, problems_cache):
    prob = problems_cache("mtb")
    orc = O.Oracle(prob)
    R, steps = 2600, 40
    sched = PB.default_schedule("mtb", n_chains=R, total_steps=steps)
    chains = sorted(set(list(range(0, R, 131)) + [1, 2, R - 1]))
    with CHandle(B, prob, sched) as hd:                                   # chains handed over between slots
        B.sa_select_kernel(hd.h, B.SA_KERNEL_DENSE)
        B.sa_set_trace(hd.h, chains, steps)
        B.sa_run(hd.h, steps)
        assert B.sa_get_info(hd.h)["grid"] < R
        check(B, hd, orc, chains, steps, B.sa_get_trace(hd.h, len(chains), steps))
    hpg = problems_cache("hpg")
    horc = O.Oracle(hpg)
    sched = PB.make_schedule(64, 5 * 40, n_levels=5)
    want = O.run_levels(horc, sched, 64, 5, 32, threads=NCPU, constrained=True)
    with CHandle(B, hpg, sched, B.SA_CONSTRAINED | B.SA_LEVEL_STATS) as hd:      # Table 1 levels, groups of 32
        B.sa_run_levels(hd.h, 5, 32)
        for c in range(64):
            cur, fc, best, fb = B.sa_get_chain(hd.h, c, hpg.n_params)
            assert np.array_equal(cur, want[c][0]) and np.array_equal(best, want[c][1]) and (fc, fb) == (want[c][2], want[c][3]), c
            assert horc.valid(cur)
        st = B.sa_get_level_stats(hd.h, 5)
        assert st["steps"].tolist() == [64 * 40] * 5


def test_large_constrained_on_the_static_kernel_and_refusals(B, problems_cache):
    prob = problems_cache("large")
    orc = O.Oracle(prob)
    sched = PB.default_schedule("large", n_chains=6, total_steps=200)
    with CHandle(B, prob, sched) as hd:
        B.sa_set_trace(hd.h, list(range(6)), 60)
        B.sa_run(hd.h, 25)
        B.sa_run(hd.h, 35)                                                # the counters are rebuilt from HBM at every launch
        assert B.sa_get_info(hd.h)["variant"] == 4                        # AUTO: the static kernel, 8 warps per chain
        check(B, hd, orc, list(range(6)), 60, B.sa_get_trace(hd.h, 6, 60))
    with pytest.raises(B.SaError):                                        # tiny has nodes without in-edges
        B.sa_create(problems_cache("tiny"), PB.default_schedule("tiny"), flags=B.SA_CONSTRAINED)


def hub_problem(n=800, hub_out=375, extra=2400, seed=77):
    """A network whose node 0 feeds `hub_out` other nodes, on a ring that gives every node an in- and an out-edge:
    enough of the hub's out-edges are non-zero in a repaired random vector for the count to pass through 257, so a
    per-node counter kept in one byte would wrap (257 reads as 1) and strike moves the oracle allows."""
    rng = np.random.default_rng(seed)
    edges = {(i, (i + 1) % n) for i in range(n)}
    edges |= {(0, int(d)) for d in rng.choice(np.arange(2, n), size=hub_out - 1, replace=False)}
    while len(edges) < n + hub_out - 1 + extra:
        s, d = (int(v) for v in rng.integers(1, n, size=2))
        if s != d:
            edges.add((s, d))
    edges = sorted(edges)
    src = np.array([e[0] for e in edges], dtype=np.int32)
    dst = np.array([e[1] for e in edges], dtype=np.int32)
    K, T = 4, 12
    times = np.array([4, 8, 12], dtype=np.int32)
    init = rng.integers(0, 3, size=(K, n)).astype(np.uint8)
    clamp = np.zeros((K, n), dtype=np.uint8)
    clamp[:, 5] = 1
    prob = PB.Problem(name="hub", seed=seed, n_nodes=n, n_edges=len(edges), edge_src=src, edge_dst=dst,
                      th_lo=np.array(PB.TH_LO, dtype=np.int8), th_hi=np.array(PB.TH_HI, dtype=np.int8), n_cond=K, n_steps=T,
                      obs_times=times, init_state=init, clamp=clamp, obs=np.full((K, len(times), n), PB.UNOBSERVED, dtype=np.uint8))
    truth = np.concatenate([rng.integers(-1, 2, size=len(edges)), rng.integers(0, len(PB.TH_LO), size=n)]).astype(np.int8)
    obs = np.asarray(O.simulate_fn(prob, truth), dtype=np.uint8).reshape(K, len(times), n).copy()
    obs[:, :, rng.choice(n, size=n // 2, replace=False)] = PB.UNOBSERVED
    prob.obs = obs
    assert int((src == 0).sum()) == hub_out
    return prob


def test_hub_with_more_than_256_out_edges_on_the_static_kernel(B):
    prob = hub_problem()
    orc = O.Oracle(prob)
    R, steps = 16, 1500
    sched = PB.make_schedule(R, steps, n_levels=10)
    hub_edges = np.nonzero(prob.edge_src == 0)[0]
    with CHandle(B, prob, sched) as hd:
        B.sa_set_trace(hd.h, list(range(R)), steps)
        B.sa_run(hd.h, steps)
        assert B.sa_get_info(hd.h)["variant"] == 4                        # N = 800: the static kernel
        refs = oracle_chains(orc, sched, list(range(R)), steps)
        # the case is only worth its name if non-zero hub edges are proposed while the hub has exactly 257 non-zero
        # out-edges (= 1 mod 256, where "to 0" would be struck by mistake): replay the oracle's traces and count
        is_hub = np.zeros(prob.n_params, dtype=bool)
        is_hub[hub_edges] = True
        hits = 0
        for c, ref in enumerate(refs):
            x = orc.init_chain(sched.seed, c, constrained=True)[0].copy()
            tr = O.unpack_trace(ref["trace"])
            count = int((x[is_hub] != 0).sum())
            for p, code, acc, null in zip(tr["param"].tolist(), tr["code"].tolist(), tr["accepted"].tolist(), tr["null_move"].tolist()):
                hits += int(is_hub[p] and x[p] != 0 and count == 257)
                if acc and not null:
                    new = code - 1 if p < prob.n_edges else code
                    if is_hub[p]:
                        count += int(new != 0) - int(x[p] != 0)
                    x[p] = new
            assert np.array_equal(x, ref["cur"])
        assert hits >= 15, hits
        check(B, hd, orc, list(range(R)), steps, B.sa_get_trace(hd.h, R, steps))
