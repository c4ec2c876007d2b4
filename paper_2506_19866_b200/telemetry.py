"""Acceptance statistics per temperature level from sa_get_trace records (
PAPER.md :235-239 discusses how often worse candidates are accepted as the temperature falls).

Pure bookkeeping over the trace records the library already writes (include/ternary_sa.h: bits
0-31 delta_cand, bit 60 accepted, bit 61 new best); no method arithmetic happens here.
"""
from __future__ import annotations

import numpy as np


def acceptance_by_level(trace: np.ndarray, init_fit, steps_per_level: int, n_levels: int, g0: int = 0) -> dict:
    """trace: [n_chains][n_steps] u64 records of steps g0 .. g0+n_steps-1; init_fit: [n_chains] the
    current fitness of each traced chain before step g0.  Returns per level (rows of the acceptance
    table, the last one absorbing steps past the schedule): steps, accepted, accepted_worse
    (accepted with delta_cand > delta_cur), improved (new best), as int64 arrays [n_levels]."""
    trace = np.atleast_2d(np.asarray(trace, dtype=np.uint64))
    n_chains, n_steps = trace.shape
    fcand = (trace & np.uint64(0xFFFFFFFF)).astype(np.int64)
    acc = ((trace >> np.uint64(60)) & np.uint64(1)).astype(bool)
    best = ((trace >> np.uint64(61)) & np.uint64(1)).astype(bool)
    cur = np.asarray(init_fit, dtype=np.int64).reshape(n_chains).copy()
    level = np.minimum((g0 + np.arange(n_steps)) // steps_per_level, n_levels - 1)
    out = {k: np.zeros(n_levels, dtype=np.int64) for k in ("steps", "accepted", "accepted_worse", "improved")}
    for s in range(n_steps):
        a = acc[:, s]
        out["steps"][level[s]] += n_chains
        out["accepted"][level[s]] += int(a.sum())
        out["accepted_worse"][level[s]] += int((a & (fcand[:, s] > cur)).sum())
        out["improved"][level[s]] += int(best[:, s].sum())
        cur = np.where(a, fcand[:, s], cur)
    out["final_fit"] = cur
    return out
