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
