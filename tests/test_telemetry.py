"""Acceptance statistics per level derived from trace records (paper_2506_19866_b200/telemetry.py)."""
import numpy as np
import pytest

from oracle import oracle as O
from paper_2506_19866_b200 import problems as PB
from paper_2506_19866_b200.telemetry import acceptance_by_level


def test_counts_match_a_replay_of_the_oracle_trace():
    prob = PB.make_problem("tiny", O.simulate_fn)
    orc = O.Oracle(prob)
    sched = PB.make_schedule(4, 400, n_levels=8)
    runs = [orc.run_chain(sched, c, 450) for c in range(4)]           # 50 steps past the schedule: level saturates
    tr = np.stack([r["trace"] for r in runs])
    st = acceptance_by_level(tr, [r["init_fit"] for r in runs], sched.steps_per_level, sched.n_levels)
    assert st["steps"].sum() == 4 * 450 and st["steps"][-1] == 4 * (50 + 50)
    assert np.array_equal(st["final_fit"], [r["fit_cur"] for r in runs])        # the replay ends where the chains did
    u = O.unpack_trace(tr)
    assert st["accepted"].sum() == int(u["accepted"].sum())
    # greedy table: nothing worse is ever accepted; always-accept table: every step is accepted
    greedy = PB.make_schedule(2, 200, n_levels=4)
    greedy.accept = np.zeros_like(greedy.accept)
    g = orc.run_chain(greedy, 0, 200)
    assert acceptance_by_level(g["trace"], [g["init_fit"]], 50, 4)["accepted_worse"].sum() == 0
    hot = PB.make_schedule(2, 200, n_levels=4, dmax=prob.n_scored)
    hot.accept = np.full((4, prob.n_scored), 0xFFFFFFFF, dtype=np.uint32)
    h = orc.run_chain(hot, 0, 200)
    s = acceptance_by_level(h["trace"], [h["init_fit"]], 50, 4)
    assert np.array_equal(s["accepted"], s["steps"]) and s["accepted_worse"].sum() > 0
    # acceptance of worse moves falls as the temperature falls (first against last level)
    many = [orc.run_chain(sched, c, 400) for c in range(4, 36)]
    m = acceptance_by_level(np.stack([r["trace"] for r in many]), [r["init_fit"] for r in many], 50, 8)
    assert m["accepted_worse"][0] > m["accepted_worse"][-1]


@pytest.mark.gpu
def test_gpu_trace_gives_the_same_statistics():
    import torch
    assert torch.cuda.is_available()
    from paper_2506_19866_b200 import binding as B
    B.use_torch_plumbing()
    prob = PB.make_problem("hpg", O.simulate_fn)
    orc = O.Oracle(prob)
    sched = PB.make_schedule(16, 600, n_levels=6)
    h = B.sa_create(prob, sched)
    try:
        f0, _ = B.sa_get_fitness(h, 16)
        B.sa_set_trace(h, list(range(16)), 600)
        B.sa_run(h, 600)
        got = acceptance_by_level(B.sa_get_trace(h, 16, 600), f0, sched.steps_per_level, sched.n_levels)
    finally:
        B.sa_destroy(h)
    runs = [orc.run_chain(sched, c, 600) for c in range(16)]
    ref = acceptance_by_level(np.stack([r["trace"] for r in runs]), [r["init_fit"] for r in runs], sched.steps_per_level, sched.n_levels)
    for k in ("steps", "accepted", "accepted_worse", "improved", "final_fit"):
        assert np.array_equal(got[k], ref[k]), k
