"""tests/resim_stats.py (the measurement behind "incremental re-simulation: does it pay?")."""
import numpy as np

from oracle import oracle as O
import resim_stats as RS
from paper_2506_19866_b200 import problems as PB


def test_counts_are_consistent_on_tiny():
    prob = PB.make_problem("tiny", O.simulate_fn)
    orc = O.Oracle(prob)
    sched = PB.make_schedule(2, 120)
    s = RS.chain_stats(prob, orc, sched, 0, 120)
    T = prob.n_steps
    assert s["first_div"].sum() == 120 and s["first_div"][0] == 0          # t = 0 is the given initial state: never differs
    assert abs(s["no_effect_frac"] - s["first_div"][T + 1] / 120) < 1e-12
    # a candidate without any effect makes every time step skippable; a skippable time step is cheap in all K conditions
    assert s["no_effect_frac"] <= s["step_skip_frac"] <= s["cheap_frac"] <= 1.0
    # every diverging candidate still enters t = 1 with the (given) initial state: at least one cheap step per condition
    assert s["cheap_frac"] >= 1.0 / T
    # all-zero weights and a threshold change of a clamped-everywhere node: no effect at all
    x = np.zeros(prob.n_params, dtype=np.int8)
    a = orc.simulate(x)
    x2 = x.copy(); x2[0] = 1                                               # an edge whose source may be active: may differ
    assert a.shape == orc.simulate(x2).shape
