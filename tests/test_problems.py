"""The seeded input generators: deterministic, structurally valid, shaped like BASELINE.json's configs."""
import numpy as np
import pytest

from oracle import oracle as O
from paper_2506_19866_b200 import problems as PB


@pytest.mark.parametrize("name", ["tiny", "hpg", "mtb", "large"])
def test_structure(problems_cache, name):
    p, spec = problems_cache(name), PB.CONFIGS[name]
    assert (p.n_nodes, p.n_edges, p.n_cond, p.n_steps) == (spec.n_nodes, spec.n_edges, spec.n_cond, spec.n_steps)
    assert p.n_params == {"tiny": 28, "hpg": 102, "mtb": 1000, "large": 11000}[name]
    assert (p.edge_src != p.edge_dst).all()                                   # no self-loops
    assert len(set(zip(p.edge_src.tolist(), p.edge_dst.tolist()))) == p.n_edges   # no duplicates
    indeg = np.bincount(p.edge_dst, minlength=p.n_nodes)
    outdeg = np.bincount(p.edge_src, minlength=p.n_nodes)
    if name != "tiny":
        assert indeg.min() >= 1 and outdeg.min() >= 1                         # closed loop
    if name == "mtb":
        assert indeg.max() <= 40
    assert (p.clamp.sum(axis=1) == spec.n_clamped).all()
    assert set(np.unique(p.init_state)) <= {0, 1, 2}
    assert set(np.unique(p.init_state[p.clamp == 1])) <= {0, 2}
    assert set(np.unique(p.obs)) <= {0, 1, 2, 255}
    n_observed = {"tiny": 4, "hpg": 10, "mtb": 56, "large": 556}[name]
    assert len(p.observed_nodes) == n_observed
    assert p.n_scored == p.n_cond * p.n_obs * n_observed
    assert int((p.obs != p.obs_clean).sum()) == p.n_flipped                   # exactly round(5 %) entries differ
    assert p.obs_times.tolist() == list(spec.obs_times)
    assert (np.diff(p.obs_times) > 0).all() and p.obs_times[0] >= 1 and p.obs_times[-1] <= p.n_steps
    assert p.node_updates_per_step == {"tiny": 192, "hpg": 1728, "mtb": 25600, "large": 512000}[name]


def test_deterministic_and_seed_sensitive():
    a = PB.make_problem("hpg", O.simulate_fn)
    b = PB.make_problem("hpg", O.simulate_fn)
    c = PB.make_problem("hpg", O.simulate_fn, seed=7)
    for f in ("edge_src", "edge_dst", "init_state", "clamp", "obs", "truth"):
        assert np.array_equal(getattr(a, f), getattr(b, f))
    assert not np.array_equal(a.edge_src, c.edge_src)


def test_schedule_defaults():
    for name, spl in (("tiny", 10), ("hpg", 100), ("mtb", 100), ("large", 5)):
        s = PB.default_schedule(name)
        assert (s.n_levels, s.dmax, s.seed) == (200, 64, 42)
        assert s.steps_per_level == spl and s.accept.shape == (200, 64) and s.accept.dtype == np.uint32
    assert PB.default_schedule("mtb", total_steps=PB.SCALING_STEPS).steps_per_level == 10


def test_spread_chains():
    ids = PB.spread_chains(4096, 32)
    assert ids[:4] == [0, 1, 2, 3] and len(ids) == 32 and ids[-1] < 4096 and ids == sorted(set(ids))
    assert PB.spread_chains(8, 32) == list(range(8))


def test_splitmix_reference_behaviour():
    r = PB.SplitMix64(1, 0)
    vals = [r.below(10) for _ in range(1000)]
    assert min(vals) == 0 and max(vals) == 9
    s = PB.SplitMix64(3, 1).sample_distinct(50, 50)
    assert sorted(s) == list(range(50))
    s = PB.SplitMix64(3, 1).sample_distinct(1000, 10)
    assert len(set(s)) == 10
