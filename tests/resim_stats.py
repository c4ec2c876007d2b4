"""Does exact incremental re-simulation pay?  (north_star: "re-simulates only the conditions reachable
from the mutated edge's target where that pays off".)

TEST / MEASUREMENT INFRASTRUCTURE: calls only oracle/ (and the shared input generators).  For SA
chains of the config model it replays every step's candidate next to the current vector and counts,
from the two full trajectories the ORACLE simulates, how much of a candidate's simulation is
identical to the current vector's and could therefore be skipped EXACTLY by a kernel that keeps the
current trajectory:

  * a (condition k, time step t) is "cheap" when the candidate's state at t-1 equals the current
    vector's state at t-1: then only the mutated node needs its sum (one row), every other node's
    new state is the stored one;
  * the kernels of this library update all K conditions of a time step together (columns of one
    MMA, byte lanes of one word), so what they can skip is a time step whose K conditions are ALL
    cheap ("step skippable");
  * "no effect": the candidate's whole trajectory equals the current one (fitness unchanged);
  * "first divergence": the first t at which any condition differs.

    python tests/resim_stats.py [--chains 3] [--steps 600]

prints one markdown table row per workload (the numbers quoted in DESIGN.md §11).
"""
from __future__ import annotations

import argparse
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from oracle import oracle as O  # noqa: E402
from paper_2506_19866_b200 import problems as PB  # noqa: E402


def chain_stats(prob, orc, sched, chain: int, n_steps: int) -> dict:
    run = orc.run_chain(sched, chain, n_steps)
    tr = O.unpack_trace(run["trace"])
    x, _ = orc.init_chain(sched.seed, chain)
    cur = orc.simulate(x)                                   # [K][T+1][N]
    K, T = prob.n_cond, prob.n_steps
    cheap = step_skip = no_effect = 0
    first_div = np.zeros(T + 2, dtype=np.int64)             # histogram over t = 1..T, T+1 = never
    reconverged = diverged = 0
    for g in range(n_steps):
        p, code = int(tr["param"][g]), int(tr["code"][g])
        cand = x.copy()
        cand[p] = code - 1 if p < prob.n_edges else code
        traj = orc.simulate(cand)
        same = (traj == cur).all(axis=2)                    # [K][T+1]: state equal at time t
        entry_same = same[:, :-1]                           # state at t-1, for t = 1..T
        cheap += int(entry_same.sum())
        step_skip += int(entry_same.all(axis=0).sum())
        if same.all():
            no_effect += 1
            first_div[T + 1] += 1
        else:
            t_first = int(np.argmax(~same.all(axis=0)))     # first time some condition differs
            first_div[t_first] += 1
            # conditions that differ at some time and are equal again at the last time point
            dk = ~same.all(axis=1)
            diverged += int(dk.sum())
            reconverged += int((dk & same[:, -1]).sum())
        if tr["accepted"][g]:
            x, cur = cand, traj
    n = n_steps
    return {"n": n, "cheap_frac": cheap / (n * K * T), "step_skip_frac": step_skip / (n * T), "no_effect_frac": no_effect / n,
            "first_div": first_div, "reconverged_frac": reconverged / max(diverged, 1),
            "accept_frac": float(tr["accepted"].mean())}


def workload_stats(name: str, chains: int, n_steps: int) -> dict:
    prob = PB.make_problem(name, O.simulate_fn)
    orc = O.Oracle(prob)
    sched = PB.make_schedule(max(chains, 1), n_steps)       # the whole cooling schedule squeezed into n_steps
    parts = [chain_stats(prob, orc, sched, c, n_steps) for c in range(chains)]
    out = {k: float(np.mean([p[k] for p in parts])) for k in ("cheap_frac", "step_skip_frac", "no_effect_frac",
                                                              "reconverged_frac", "accept_frac")}
    hist = sum(p["first_div"] for p in parts)
    T = prob.n_steps
    out["first_div_median"] = int(np.searchsorted(np.cumsum(hist), hist.sum() / 2) )
    out["first_div_le_2"] = float(hist[:3].sum() / hist.sum())
    out["T"] = T
    out["name"] = name
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--chains", type=int, default=3)
    ap.add_argument("--steps", type=int, default=600)
    ap.add_argument("--workloads", default="hpg,mtb,large")
    args = ap.parse_args()
    print("| workload | accepted | candidates with no effect at all | (k, t) pairs entered with an unchanged state | time steps with ALL K conditions unchanged (what the kernels could skip) | first divergence at t <= 2 | diverged conditions equal again at t = T |")
    print("|---|---|---|---|---|---|---|")
    for name in args.workloads.split(","):
        steps = args.steps if name != "large" else max(60, args.steps // 5)
        s = workload_stats(name, args.chains, steps)
        print(f"| {name} ({args.chains} chains x {steps} steps) | {s['accept_frac']:.2f} | {s['no_effect_frac']:.3f} | {s['cheap_frac']:.3f} | "
              f"{s['step_skip_frac']:.3f} | {s['first_div_le_2']:.3f} | {s['reconverged_frac']:.3f} |")


if __name__ == "__main__":
    main()
