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


FAMILIES = [("hpg", "GENERIC", {}), ("hpg", "GENERIC", {"TSA_KERNEL": "cta"}), ("hpg", "STATIC", {}), ("hpg", "DENSE", {}),
            ("mtb", "DENSE", {}), ("mtb", "STATIC", {})]


@pytest.mark.gpu
@pytest.mark.parametrize("name,family,env", FAMILIES, ids=[f"{n}-{f}-{'-'.join(e.values()) or 'default'}" for n, f, e in FAMILIES])
def test_device_level_statistics_of_every_kernel_family(name, family, env):
    """sa_get_level_stats (SA_LEVEL_STATS): counters kept by the kernels themselves, per temperature level,
    equal to the statistics of the traced records of the same run and to those of the oracle's traces
    (PAPER.md:237); steps past the schedule land in the last row; several sa_run calls add up."""
    import os
    import torch
    assert torch.cuda.is_available()
    from paper_2506_19866_b200 import binding as B
    B.use_torch_plumbing()
    prob = PB.make_problem(name, O.simulate_fn)
    orc = O.Oracle(prob)
    R, L, spl = 40, 6, 50
    sched = PB.make_schedule(R, L * spl, n_levels=L)
    n = L * spl + 35
    os.environ.update(env)
    try:
        h = B.sa_create(prob, sched, flags=B.SA_LEVEL_STATS)
        try:
            B.sa_select_kernel(h, getattr(B, "SA_KERNEL_" + family))
            f0, _ = B.sa_get_fitness(h, R)
            B.sa_set_trace(h, list(range(R)), n)
            B.sa_run(h, 77)
            B.sa_run(h, n - 77)
            got = B.sa_get_level_stats(h, L)
            tr = B.sa_get_trace(h, R, n)
        finally:
            B.sa_destroy(h)
    finally:
        for k in env:
            del os.environ[k]
    from_trace = acceptance_by_level(tr, f0, spl, L)
    runs = [orc.run_chain(sched, c, n) for c in range(R)]
    ref = acceptance_by_level(np.stack([r["trace"] for r in runs]), [r["init_fit"] for r in runs], spl, L)
    for k in ("steps", "accepted", "accepted_worse", "improved"):
        assert np.array_equal(got[k], from_trace[k]), k
        assert np.array_equal(got[k], ref[k]), k
    assert got["steps"].tolist() == [R * spl] * (L - 1) + [R * (spl + 35)]


@pytest.mark.gpu
def test_level_statistics_with_balanced_slots_and_without_the_flag():
    """More chains than resident slots: chains are cut into pieces that run in different slots; the
    counters still add up to steps x chains per level.  Without SA_LEVEL_STATS the call refuses."""
    import torch
    assert torch.cuda.is_available()
    from paper_2506_19866_b200 import binding as B
    B.use_torch_plumbing()
    prob = PB.make_problem("mtb", O.simulate_fn)
    R, L, spl = 2600, 4, 11
    sched = PB.make_schedule(R, L * spl, n_levels=L)
    h = B.sa_create(prob, sched, flags=B.SA_LEVEL_STATS)
    try:
        B.sa_select_kernel(h, B.SA_KERNEL_DENSE)
        B.sa_set_trace(h, list(range(0, R, 100)), L * spl)
        f0, _ = B.sa_get_fitness(h, R)
        B.sa_run(h, L * spl)
        got = B.sa_get_level_stats(h, L)
        assert B.sa_get_info(h)["grid"] < R                               # balanced slots were used
        tr = B.sa_get_trace(h, len(range(0, R, 100)), L * spl)
    finally:
        B.sa_destroy(h)
    assert got["steps"].tolist() == [R * spl] * L
    sub = acceptance_by_level(tr, f0[::100], spl, L)
    assert (got["accepted"] >= sub["accepted"]).all() and (got["accepted"] <= got["steps"]).all()
    h = B.sa_create(prob, PB.make_schedule(8, 40, n_levels=4))
    try:
        with pytest.raises(B.SaError):
            B.sa_get_level_stats(h, 4)
    finally:
        B.sa_destroy(h)
