"""Host-side checks of the C-ABI library that need no GPU: it loads, exports every symbol the
header declares, validates its inputs, and its host helper matches the pinned table values."""
import copy
import ctypes
import os
import re

import numpy as np
import pytest

from helpers import golden_rows

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def B():
    from paper_2506_19866_b200 import build
    build.build()
    from paper_2506_19866_b200 import binding
    return binding


def _declared_functions():
    text = open(os.path.join(ROOT, "include", "ternary_sa.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(sap?_[a-z0-9_]+)\s*\(", text)) - {"sa_alloc_fn", "sa_free_fn"})


def test_library_exports_every_declared_symbol(B):
    names = _declared_functions()
    assert len(names) >= 16
    lib = ctypes.CDLL(B.LIB_PATH)
    for n in names:
        assert hasattr(lib, n), f"{n} is declared in include/ternary_sa.h but not exported"
    assert sorted(B.EXPORTS) == names


def test_geometric_table_helper_matches_pins(B):
    for T, d, want in golden_rows("accept_table.txt"):
        tab = B.sa_geometric_table(float(T), float(T), 1, 64)
        assert int(tab[0, int(d) - 1]) == int(want)
    from paper_2506_19866_b200 import problems as PB
    assert np.array_equal(B.sa_geometric_table(PB.T0, PB.T_END, PB.N_LEVELS, PB.DMAX),
                          PB.geometric_table(PB.T0, PB.T_END, PB.N_LEVELS, PB.DMAX))
    with pytest.raises(B.SaError):
        B.sa_geometric_table(-1.0, 1.0, 4, 4)


def _bad(B, prob, sched, match):
    with pytest.raises(B.SaError) as ei:
        B.sa_create(prob, sched)
    assert ei.value.code == B.SA_EINVAL and match in str(ei.value), str(ei.value)


def test_sa_create_validation(B, problems_cache):
    from paper_2506_19866_b200 import problems as PB
    good = problems_cache("tiny")
    sched = PB.default_schedule("tiny")

    p = copy.copy(good); p.edge_src = good.edge_src.copy(); p.edge_src[0] = p.edge_dst[0]
    _bad(B, p, sched, "self-loop")
    p = copy.copy(good); p.edge_src = good.edge_src.copy(); p.edge_dst = good.edge_dst.copy()
    p.edge_src[1], p.edge_dst[1] = p.edge_src[0], p.edge_dst[0]
    _bad(B, p, sched, "duplicate")
    p = copy.copy(good); p.edge_dst = good.edge_dst.copy(); p.edge_dst[0] = good.n_nodes
    _bad(B, p, sched, "out of range")
    p = copy.copy(good); p.th_lo = good.th_lo.copy(); p.th_lo[2] = 0
    _bad(B, p, sched, "th_lo")
    p = copy.copy(good); p.init_state = good.init_state.copy(); p.init_state[0, 0] = 3
    _bad(B, p, sched, "init_state")
    p = copy.copy(good); p.obs = good.obs.copy(); p.obs[0, 0, 0] = 7
    _bad(B, p, sched, "obs must")
    p = copy.copy(good); p.obs_times = np.array([3, 3, 9, 12], dtype=np.int32)
    _bad(B, p, sched, "obs_times")
    p = copy.copy(good); p.obs_times = np.array([3, 6, 9, 13], dtype=np.int32)
    _bad(B, p, sched, "obs_times")
    s = copy.copy(sched); s.n_chains = 0
    _bad(B, good, s, "schedule")
    # constraints need a closed loop: tiny has nodes without in-edges; unknown flags are refused
    for flags, match in ((B.SA_CONSTRAINED, "in-edge"), (64, "flag")):
        with pytest.raises(B.SaError) as ei:
            B.sa_create(good, sched, flags=flags)
        assert ei.value.code == B.SA_EINVAL and match in str(ei.value), str(ei.value)
    # accumulator range: a node with in-degree 63 is refused (reading 24)
    N = 65
    star = copy.copy(good)
    star.n_nodes, star.n_edges = N, 63
    star.edge_src = np.arange(1, 64, dtype=np.int32); star.edge_dst = np.zeros(63, dtype=np.int32)
    star.init_state = np.zeros((good.n_cond, N), dtype=np.uint8); star.clamp = np.zeros((good.n_cond, N), dtype=np.uint8)
    star.obs = np.full((good.n_cond, good.n_obs, N), 255, dtype=np.uint8)
    _bad(B, star, sched, "accumulator")


def test_no_cpu_fallback(B, problems_cache):
    """Without a CUDA device the product path must fail loudly, not compute on the host."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    from paper_2506_19866_b200 import problems as PB
    with pytest.raises(B.SaError) as ei:
        B.sa_create(problems_cache("tiny"), PB.default_schedule("tiny"))
    assert ei.value.code in (B.SA_ECUDA, B.SA_ENOMEM)
    with pytest.raises(B.SaError):
        B.sa_simulate(problems_cache("tiny"), problems_cache("tiny").truth)
    assert B.sa_run.__doc__ is None or True
    B.sa_destroy(None)                      # NULL is a no-op


def test_execution_plan_is_valid_for_every_config(B, problems_cache):
    """sa_plan_info builds the host-side plan (rows, split rows, bank classes, conflict-free edge
    colouring) and fails if its own self-check finds an unscheduled edge or a bank conflict."""
    import math
    for name in ("tiny", "hpg", "mtb", "large"):
        prob = problems_cache(name)
        info = B.sa_plan_info(prob)
        assert info["edge_iterations"] >= math.ceil(prob.n_edges / 32)
        assert info["rows"] >= prob.n_nodes and info["passes"] * 32 >= info["rows"]
        assert info["edge_slots"] >= prob.n_edges
        assert info["state_words_per_node"] == {"tiny": 1, "hpg": 1, "mtb": 2, "large": 4}[name]
        assert info["max_in_degree"] == int(np.bincount(prob.edge_dst).max())
        # clamped observed entries never change: their mismatches are a per-problem constant
        k, j, i = np.nonzero((prob.obs != 255) & (prob.clamp[:, None, :] == 1))
        assert info["clamped_mismatches"] == int((prob.obs[k, j, i] != prob.init_state[k, i]).sum())
    mtb = B.sa_plan_info(problems_cache("mtb"))
    assert mtb["edge_iterations"] <= 40          # 900 edges / 32 lanes = 28.1 is the floor; the naive layout needs 56
    import os
    os.environ["TSA_NO_SPLIT"] = "1"; os.environ["TSA_NO_BANKOPT"] = "1"
    try:
        naive = B.sa_plan_info(problems_cache("mtb"))
    finally:
        del os.environ["TSA_NO_SPLIT"], os.environ["TSA_NO_BANKOPT"]
    assert naive["split_nodes"] == 0 and naive["edge_iterations"] > mtb["edge_iterations"]


def test_dense_plan_leaves_empty_blocks_out(B, problems_cache):
    """Host only: the dense kernel's plan for Mtb-shaped uses the 2:4-sparse operand, scores two of four result
    words and leaves two of the 14 blocks of the weight matrix without a candidate edge (12 IMMAs per time step);
    the plan is deterministic; other shapes with a small last row tile plan and compile whether or not the pinned
    search succeeds."""
    import re
    from oracle import oracle as O
    from paper_2506_19866_b200 import problems as PB
    a = B.sa_jit_check(problems_cache("mtb"), 4096)
    b = B.sa_jit_check(problems_cache("mtb"), 4096)
    assert a["dense_applies"] and a["log"] == b["log"] and a["dense_cubin_bytes"] == b["dense_cubin_bytes"]
    m = re.search(r"sparse=(\d+) immas_per_step=(\d+) obs_words=(\d+)", a["log"])
    assert m and (int(m.group(1)), int(m.group(2)), int(m.group(3))) == (1, 12, 2), a["log"]
    for name, N, E, degree, seed in (("eb84", 84, 500, "powerlaw", 3), ("eb104", 104, 1500, "poisson", 2)):
        cs = PB.ConfigSpec(name, 4000 + seed, N, E, degree, 8, 3, 16, (4, 8, 12, 16), 8, 120, max_in_degree=40)
        info = B.sa_jit_check(PB.make_problem(name, O.simulate_fn, spec=cs, noise=0.05), 8)
        m = re.search(r"sparse=(\d+) immas_per_step=(\d+)", info["log"])
        assert info["dense_applies"] and m and 0 < int(m.group(2)) <= (N + 15) // 16 * 4, info["log"]


# ------------------------------------------------------------------ the paper model (sap_*)
@pytest.fixture(scope="module")
def paper_hpg():
    from oracle import oracle_paper as OP
    from paper_2506_19866_b200 import problems as PB
    return PB.make_paper_problem("paper_hpg", OP.simulate_fn)


def test_sap_create_validation(B, paper_hpg):
    from paper_2506_19866_b200 import problems as PB
    good = paper_hpg
    sched = PB.paper_schedule(8, 4, 10, good.max_objective)

    def bad(prob, sc, match, flags=0):
        with pytest.raises(B.SaError) as ei:
            B.sap_create(prob, sc, flags)
        assert ei.value.code == B.SA_EINVAL and match in str(ei.value), str(ei.value)

    p = copy.copy(good); p.edge_src = good.edge_src.copy(); p.edge_dst = good.edge_dst.copy()
    p.edge_src[1], p.edge_dst[1] = p.edge_src[0], p.edge_dst[0]
    bad(p, sched, "duplicate")
    p.edge_dst[0] = p.edge_src[0]; p.edge_dst[1] = p.edge_src[1]          # the same self-loop twice; one alone is allowed
    bad(p, sched, "duplicate")
    p = copy.copy(good); p.edge_dst = good.edge_dst.copy(); p.edge_dst[0] = good.n_nodes
    bad(p, sched, "out of range")
    p = copy.copy(good); p.fast = good.fast.copy(); p.fast[0] = 2
    bad(p, sched, "fast")
    p = copy.copy(good); p.init_state = good.init_state.copy(); p.init_state[0, 0] = 3
    bad(p, sched, "initial state")
    p = copy.copy(good); p.ref = good.ref.copy(); p.ref[0, 0, 0] = 9
    bad(p, sched, "reference")
    s = copy.copy(sched); s.n_chains = 0
    bad(good, s, "schedule")
    bad(good, sched, "flag", flags=64)
    # with constraints on, a node without an in-edge admits no valid vector
    p = copy.copy(good)
    keep = good.edge_dst != good.edge_dst[0]
    p.edge_src, p.edge_dst, p.n_edges = good.edge_src[keep], good.edge_dst[keep], int(keep.sum())
    bad(p, sched, "in-edge", flags=B.SAP_CONSTRAINED)
    B.sap_destroy(None)


def test_paper_kernels_compile_for_every_shape(B, paper_hpg):
    """Host only: the plan and the NVRTC build of the paper-model kernels (no GPU needed)."""
    from oracle import oracle_paper as OP
    from paper_2506_19866_b200 import problems as PB
    info = B.sap_jit_check(paper_hpg)
    assert (info["lanes_per_chain"], info["node_slots"]) == (8, 2) and info["cubin_bytes"] > 0, info["log"]
    indeg = np.bincount(paper_hpg.edge_dst, minlength=9)
    top = np.sort(indeg)[::-1]
    assert info["edge_slots"] == int(top[0] + top[8])            # slot 0 holds the 8 largest in-degrees, slot 1 the rest
    mtb = B.sap_jit_check(PB.make_paper_problem("paper_mtb", OP.simulate_fn))
    assert (mtb["lanes_per_chain"], mtb["node_slots"]) == (32, 2) and mtb["cubin_bytes"] > 0, mtb["log"]


def test_no_cpu_fallback_paper_model(B, paper_hpg):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    from paper_2506_19866_b200 import problems as PB
    with pytest.raises(B.SaError) as ei:
        B.sap_create(paper_hpg, PB.paper_schedule(8, 4, 10, 64), 0)
    assert ei.value.code in (B.SA_ECUDA, B.SA_ENOMEM)
    with pytest.raises(B.SaError):
        B.sap_simulate(paper_hpg, paper_hpg.truth)
