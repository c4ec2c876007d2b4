"""sa_level_sync_static: the level synchronisation for callers that may not allocate device memory.

Some users of this library cannot call cudaMalloc once their set-up is over: they share the GPU with a framework that
has already reserved all of its memory, their own arena is frozen after start-up, or their service loop cannot take the
device-wide stall an allocation implies.  sa_run_levels allocates its winner table on a handle's first call, so it is
closed to them; sa_level_sync_static keeps that table in a fixed array inside the library (at most
SA_LEVEL_SYNC_STATIC_MAX_GROUPS groups) and allocates nothing.

The checks here: driving Table 1 as { sa_run; sa_level_sync_static } leaves every chain exactly (bit for bit, the bar of
every parity test in this repository) as the existing sa_run_levels does, on two levels in a row and with group counts
that shrink and grow between calls (the array keeps the last call's winners); sizes beyond the array are refused with a
message that names the limit.  The file sorts last on purpose: `pytest -x` stops at the first failure, and a failure in
this extra entry point must not hide the parity tests of the hot path.
"""
import numpy as np
import pytest

from oracle import oracle as O
from paper_2506_19866_b200 import problems as PB


@pytest.fixture(scope="module")
def B():
    import torch
    assert torch.cuda.is_available(), "the gpu tests need a CUDA device"
    from paper_2506_19866_b200 import build
    build.build()
    from paper_2506_19866_b200 import binding
    binding.use_torch_plumbing()
    return binding


def chain_store(B, h, R, n_params):
    fc, fb = B.sa_get_fitness(h, R)
    rows = [B.sa_get_chain(h, c, n_params) for c in range(R)]
    return fc, fb, rows


@pytest.mark.gpu
@pytest.mark.parametrize("name,R,spl,groups", [("hpg", 96, 25, (7, 0)), ("hpg", 96, 25, (0, 1, 32)), ("tiny", 8, 10, (1, 1)),
                                               ("mtb", 40, 15, (32, 7)), ("mtb", 300, 6, (256, 300)), ("large", 6, 5, (0, 4))])
def test_static_level_sync_equals_sa_run_levels(B, name, R, spl, groups):
    prob = PB.make_problem(name, O.simulate_fn)
    sched = PB.make_schedule(R, len(groups) * spl, n_levels=len(groups))
    assert sched.steps_per_level == spl
    ha, hb = B.sa_create(prob, sched), B.sa_create(prob, sched)
    try:
        for level, group in enumerate(groups):
            B.sa_run_levels(ha, 1, group)                     # the existing path: allocates its winner table on first use
            B.sa_run(hb, spl)
            B.sa_level_sync_static(hb, group)                 # the path under test: no allocation
            fca, fba, rows_a = chain_store(B, ha, R, prob.n_params)
            fcb, fbb, rows_b = chain_store(B, hb, R, prob.n_params)
            assert np.array_equal(fca, fcb) and np.array_equal(fba, fbb), f"level {level}: fitnesses"
            for c in range(R):
                (cur_a, f1a, best_a, f2a), (cur_b, f1b, best_b, f2b) = rows_a[c], rows_b[c]
                assert (f1a, f2a) == (f1b, f2b), f"level {level} chain {c}: fitness"
                assert np.array_equal(cur_a, cur_b) and np.array_equal(best_a, best_b), f"level {level} chain {c}: vectors"
            # and the synchronisation did what Table 1 says: inside a group everybody holds the group's best
            g = R if group == 0 or group > R else group
            for first in range(0, R, g):
                members = range(first, min(R, first + g))
                assert len({int(fbb[c]) for c in members}) == 1 and all(fcb[c] == fbb[c] for c in members)
                assert all(np.array_equal(rows_b[c][0], rows_b[first][2]) for c in members)
    finally:
        B.sa_destroy(ha)
        B.sa_destroy(hb)


@pytest.mark.gpu
def test_static_level_sync_refuses_more_groups_than_its_table(B):
    prob = PB.make_problem("tiny", O.simulate_fn)
    R = B.SA_LEVEL_SYNC_STATIC_MAX_GROUPS + 5
    sched = PB.make_schedule(R, 8, n_levels=2)
    h = B.sa_create(prob, sched)
    try:
        B.sa_run(h, 4)
        before = B.sa_get_fitness(h, R)[0].copy()
        with pytest.raises(B.SaError) as err:
            B.sa_level_sync_static(h, 1)                      # R groups of one chain: 5 too many
        assert str(B.SA_LEVEL_SYNC_STATIC_MAX_GROUPS) in str(err.value) and "groups" in str(err.value)
        with pytest.raises(B.SaError):
            B.sa_level_sync_static(h, -1)
        assert np.array_equal(B.sa_get_fitness(h, R)[0], before), "a refused call must not touch the chains"
        B.sa_level_sync_static(h, 2)                          # (R + 1) / 2 groups fit
        B.sa_level_sync_static(h, 0)                          # one group: everybody gets the overall best
        fc, fb = B.sa_get_fitness(h, R)
        assert fc.min() == fc.max() == fb.min() == fb.max()
        fit, chain, params = B.sa_best(h, prob.n_params)
        assert fit == fb[0] and O.Oracle(prob).fitness(params) == fit
    finally:
        B.sa_destroy(h)
