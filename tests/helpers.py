"""Shared test helpers: hand-specified example networks and golden-file readers."""
import functools
import os
import subprocess
import tempfile

import numpy as np

from paper_2506_19866_b200 import problems as PB

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def golden_rows(name):
    rows = []
    with open(os.path.join(GOLDEN, name)) as f:
        for line in f:
            line = line.strip()
            if line and not line.startswith("#"):
                rows.append(line.split())
    return rows


def example_problem(with_condition_b=False):
    """The 3-node network of SURVEY.md §8(c) Pins 1-2 (tests/golden/example_*.txt headers)."""
    src = np.array([1, 2, 0, 2, 0, 1], dtype=np.int32)
    dst = np.array([0, 0, 1, 1, 2, 2], dtype=np.int32)
    truth = np.array([-1, +1, +1, -1, -1, +1, 0, 3, 2], dtype=np.int8)
    if not with_condition_b:
        K, T, times = 1, 6, [1, 2, 3, 4, 5, 6]
        init = np.array([[0, 1, 2]], dtype=np.uint8)
        clamp = np.zeros((1, 3), dtype=np.uint8)
        obs = np.full((1, 6, 3), 255, dtype=np.uint8)
    else:
        K, T, times = 2, 6, [2, 4, 6]
        init = np.array([[0, 1, 2], [0, 1, 2]], dtype=np.uint8)
        clamp = np.array([[0, 0, 0], [0, 0, 1]], dtype=np.uint8)
        U = 255
        obs = np.array([[[2, 1, U], [1, 1, U], [2, 1, U]],
                        [[2, 1, U], [0, 1, U], [2, 1, U]]], dtype=np.uint8)   # cond 1, t=4, node 0: 2 -> 0
    return PB.Problem(name="example", seed=0, n_nodes=3, n_edges=6, edge_src=src, edge_dst=dst,
                      th_lo=np.array(PB.TH_LO, dtype=np.int8), th_hi=np.array(PB.TH_HI, dtype=np.int8),
                      n_cond=K, n_steps=T, obs_times=np.array(times, dtype=np.int32),
                      init_state=init, clamp=clamp, obs=obs, truth=truth)


def brute_force_problem(simulate, seed=77):
    """4 nodes, 6 edges, K=2, T=6: small enough to enumerate all 3^6 * 6^4 = 944 784 settings."""
    spec = PB.ConfigSpec("bf4", seed, 4, 6, "uniform-pairs", 2, 1, 6, (2, 4, 6), 4, 100)
    return PB.make_problem("bf4", simulate, spec=spec, noise=0.0)


def all_settings(n_edges, n_nodes, n_pairs):
    """Every parameter vector, int8 [3^E * n_pairs^N][E+N], edge 0 fastest."""
    total = 3 ** n_edges * n_pairs ** n_nodes
    idx = np.arange(total, dtype=np.int64)
    out = np.zeros((total, n_edges + n_nodes), dtype=np.int8)
    for e in range(n_edges):
        out[:, e] = (idx % 3) - 1
        idx //= 3
    for i in range(n_nodes):
        out[:, n_edges + i] = idx % n_pairs
        idx //= n_pairs
    return out


_ATEN_SRC = r"""
#include <ATen/core/PhiloxRNGEngine.h>
#include <cstdio>
#include <cstdlib>
int main() {
  unsigned long long seed, sub, off;
  while (scanf("%llu %llu %llu", &seed, &sub, &off) == 3) {
    at::Philox4_32 eng(seed, sub, off);
    unsigned r0 = eng(), r1 = eng(), r2 = eng(), r3 = eng();
    printf("%u %u %u %u\n", r0, r1, r2, r3);
  }
  return 0;
}
"""


@functools.lru_cache(maxsize=1)
def _aten_philox_exe():
    """ATen's own Philox4_32 engine compiled into a tiny program: an implementation of Philox4x32-10
    that is independent of the oracle's and of the CUDA path's (SURVEY.md §8(c) Pin 8)."""
    import torch
    inc = os.path.join(os.path.dirname(torch.__file__), "include")
    td = tempfile.mkdtemp(prefix="aten_philox_")
    src, exe = os.path.join(td, "p.cpp"), os.path.join(td, "p")
    with open(src, "w") as f:
        f.write(_ATEN_SRC)
    subprocess.check_call(["g++", "-O1", "-std=c++17", "-I", inc, src, "-o", exe])
    return exe


def aten_philox_blocks(cases):
    """cases: (seed, subsequence, offset) triples -> one [r0, r1, r2, r3] block each, from
    at::Philox4_32(seed, subsequence, offset).  Correspondence with the method's counter layout:
    subsequence = chain | domain << 32, offset = step g (checked by test_philox_matches_aten_engine)."""
    text = "".join(f"{s} {sub} {off}\n" for s, sub, off in cases)
    out = subprocess.check_output([_aten_philox_exe()], input=text.encode()).decode().split("\n")
    return [[int(v) for v in line.split()] for line in out if line.strip()]
