"""The level structure of PAPER.md Table 1 (:125-155): oracle pins (CPU) and GPU parity of
sa_run_levels (device-side synchronisation)."""
import copy

import numpy as np
import pytest

from oracle import oracle as O
from paper_2506_19866_b200 import problems as PB


@pytest.fixture(scope="module")
def tiny():
    return PB.make_problem("tiny", O.simulate_fn)


def test_after_a_level_every_member_holds_the_group_minimum(tiny):
    """:150-153: d*_best = min over the threads; every x_best = x*_best.  Checked against a plain
    recomputation from independently advanced chains (Oracle.run_chain is pinned elsewhere)."""
    orc = O.Oracle(tiny)
    sched = PB.make_schedule(8, 400, n_levels=10)          # 10 levels x 40 steps
    for group in (0, 4, 3):
        states = O.run_levels(orc, sched, 8, 1, group)
        solo = [orc.run_chain(sched, c, 40, trace=False) for c in range(8)]       # level 1 of fresh chains
        size = 8 if group == 0 else group
        for first in range(0, 8, size):
            members = list(range(first, min(8, first + size)))
            fits = [solo[c]["fit_best"] for c in members]
            star = members[int(np.argmin(fits))]                                    # argmin returns the first minimum
            for c in members:
                cur, best, fc, fb = states[c]
                assert fc == fb == min(fits)
                assert np.array_equal(best, solo[star]["best"]) and np.array_equal(cur, best)
                assert orc.fitness(best) == fb


def test_best_is_broadcast_not_current_and_ties_go_to_the_smallest_chain(tiny):
    """Nothing observed: every fitness is 0, so no chain ever improves strictly, each x_best stays the
    initial vector while x_current random-walks (d = 0 is accepted, reading 1), and all ties resolve to
    chain 0: after one level every chain must hold chain 0's INITIAL vector."""
    blind = copy.copy(tiny)
    blind.obs = np.full_like(tiny.obs, 255)
    orc = O.Oracle(blind)
    sched = PB.make_schedule(5, 200, n_levels=10)          # 10 levels x 20 steps
    x0, f0 = orc.init_chain(sched.seed, 0)
    assert f0 == 0
    walked = orc.run_chain(sched, 0, 20, trace=False)
    assert not np.array_equal(walked["cur"], x0)                                   # the current vector did move
    for cur, best, fc, fb in O.run_levels(orc, sched, 5, 1, 0):
        assert np.array_equal(best, x0) and np.array_equal(cur, x0) and fc == fb == 0


def test_levels_compose_and_the_global_best_never_gets_worse(tiny):
    orc = O.Oracle(tiny)
    sched = PB.make_schedule(6, 200, n_levels=20)          # 20 levels x 10 steps
    a = O.run_levels(orc, sched, 6, 7, 0)
    b = O.run_levels(orc, sched, 6, 3, 0)
    b = O.run_levels(orc, sched, 6, 4, 0, g0=30, states=b)                         # 3 + 4 levels == 7 levels
    for (c1, b1, f1, g1), (c2, b2, f2, g2) in zip(a, b):
        assert np.array_equal(c1, c2) and np.array_equal(b1, b2) and (f1, g1) == (f2, g2)
    prev = None
    for n in range(1, 8):
        fb = O.run_levels(orc, sched, 6, n, 0)[0][3]
        assert prev is None or fb <= prev
        prev = fb
    # groups of one chain: no exchange, only x_current = x_best at every level (:129)
    solo = O.run_levels(orc, sched, 6, 2, 1)
    for c in range(6):
        s1 = orc.run_chain(sched, c, 10, trace=False)
        s2 = orc.run_chain(sched, c, 10, g0=10, state=(s1["best"], s1["best"], s1["fit_best"], s1["fit_best"]), trace=False)
        assert np.array_equal(solo[c][1], s2["best"]) and solo[c][3] == s2["fit_best"]


# ------------------------------------------------------------------------------------ GPU
@pytest.fixture(scope="module")
def B():
    import torch
    assert torch.cuda.is_available(), "the gpu tests need a CUDA device"
    from paper_2506_19866_b200 import build
    build.build()
    from paper_2506_19866_b200 import binding
    binding.use_torch_plumbing()
    return binding


@pytest.mark.gpu
@pytest.mark.parametrize("name,R,levels,spl,group", [("tiny", 8, 12, 10, 0), ("hpg", 96, 6, 25, 0), ("hpg", 96, 6, 25, 32),
                                                     ("mtb", 40, 4, 15, 0), ("mtb", 40, 4, 15, 7), ("large", 6, 2, 5, 0)])
def test_sa_run_levels_matches_the_oracle(B, name, R, levels, spl, group):
    prob = PB.make_problem(name, O.simulate_fn)
    orc = O.Oracle(prob)
    sched = PB.make_schedule(R, levels * spl, n_levels=levels)
    assert sched.steps_per_level == spl
    ref = O.run_levels(orc, sched, R, levels, group, threads=8)
    h = B.sa_create(prob, sched)
    try:
        B.sa_run_levels(h, levels - 1, group)
        B.sa_run_levels(h, 1, group)
        fc, fb = B.sa_get_fitness(h, R)
        for c in range(R):
            cur, f1, best, f2 = B.sa_get_chain(h, c, prob.n_params)
            assert (f1, f2) == (ref[c][2], ref[c][3]) == (fc[c], fb[c]), f"chain {c} fitness"
            assert np.array_equal(cur, ref[c][0]) and np.array_equal(best, ref[c][1]), f"chain {c} vectors"
        B.sa_run(h, 3)                                       # off a level boundary now
        with pytest.raises(B.SaError):
            B.sa_run_levels(h, 1, group)
    finally:
        B.sa_destroy(h)
