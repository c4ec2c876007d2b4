"""The N > 1 plumbing of bench.py on CPU (gloo, world size 2): chain-range partition by rank,
max-over-ranks timing, rank 0 alone reports.  The data path has no collective."""
import json
import os
import subprocess
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import json, os, sys
sys.path.insert(0, {root!r})
import numpy as np
import torch
import torch.distributed as dist
import bench
from oracle import oracle as O
from paper_2506_19866_b200 import problems as PB

dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
chains = 3
prob = PB.make_problem("tiny", O.simulate_fn)
sched = PB.make_schedule(chains, 200, chain_id_base=bench.rank_chain_base(rank, chains))
orc = O.Oracle(prob)
fits = [orc.run_chain(sched, c + sched.chain_id_base, 200)["fit_best"] for c in range(chains)]
mine = torch.tensor(fits, dtype=torch.int64)
gathered = [torch.zeros_like(mine) for _ in range(world)]
dist.all_gather(gathered, mine)
ms = bench.max_over_ranks(10.0 + 5.0 * rank, dist, device="cpu")
if rank == 0:
    print(json.dumps({{"fits": torch.cat(gathered).tolist(), "ms": ms, "world": world}}))
dist.barrier()
dist.destroy_process_group()
"""


def test_two_rank_partition_and_timing(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER.format(root=ROOT))
    env = dict(os.environ, MASTER_ADDR="127.0.0.1")
    out = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
                          "--master-addr", "127.0.0.1", "--master-port", "29671", str(script)],
                         capture_output=True, text=True, timeout=600, env=env, cwd=ROOT)
    assert out.returncode == 0, out.stderr[-2000:]
    line = [l for l in out.stdout.splitlines() if l.startswith("{")][-1]
    got = json.loads(line)
    assert got["world"] == 2 and got["ms"] == 15.0          # the slowest rank sets the time
    # the two ranks' chains are global chains 0..5 of one 6-chain run
    sys.path.insert(0, ROOT)
    from oracle import oracle as O
    from paper_2506_19866_b200 import problems as PB
    prob = PB.make_problem("tiny", O.simulate_fn)
    sched = PB.make_schedule(6, 200)
    orc = O.Oracle(prob)
    ref = [orc.run_chain(sched, c, 200)["fit_best"] for c in range(6)]
    assert got["fits"] == ref


def test_reference_arm_prints_on_rank0_only():
    env = dict(os.environ, MASTER_ADDR="127.0.0.1")
    out = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
                          "--master-addr", "127.0.0.1", "--master-port", "29672", os.path.join(ROOT, "bench.py"),
                          "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "0", "--workload", "tiny"],
                         capture_output=True, text=True, timeout=600, env=env, cwd=ROOT)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [l for l in out.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["value"] > 0 and d["cpu_baseline"]["kind"] == "oracle"


def test_gpus_flag_without_torchrun():
    """`python bench.py --gpus 2` as the driver runs it, with no torchrun environment: the reference arm
    runs in this one process and reports n_gpus = 2; our arm starts two ranks itself, and on a box
    without two CUDA devices each of them fails loudly instead of measuring one GPU as if it were two."""
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "WORLD_SIZE", "LOCAL_RANK")}
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1",
                          "--warmup", "0", "--workload", "paper_hpg"], capture_output=True, text=True, timeout=600, env=env, cwd=ROOT)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [l for l in out.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["value"] > 0 and "paper model" in d["config"]["workload"]
    import torch
    if torch.cuda.is_available() and torch.cuda.device_count() >= 2:
        return
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--steps", "1", "--warmup", "0",
                          "--workload", "tiny", "--no-extra"], capture_output=True, text=True, timeout=600, env=env, cwd=ROOT)
    assert out.returncode != 0
    assert not [l for l in out.stdout.splitlines() if l.startswith("{")]          # no bench line from a run that cannot be N = 2
    assert "CUDA device" in out.stderr or "CUDA devices" in out.stderr


def test_instruction_counts_file_names_existing_captures():
    """profiles/inst_counts.json (the per-kernel instruction counts bench.py turns into the issue-slot
    fraction) cites capture summaries that exist under profiles/."""
    with open(os.path.join(ROOT, "profiles", "inst_counts.json")) as f:
        counts = json.load(f)
    assert "mtb" in counts
    for name, c in counts.items():
        if name.startswith("_"):
            continue
        assert c["warp_inst_per_chain_step"] > 0 and c["kernel"]
        cited = c["source"].split()[0]
        assert os.path.exists(os.path.join(ROOT, cited)), cited


def test_instruction_counts_belong_to_the_kernels_in_the_tree():
    """Every entry of profiles/inst_counts.json records the source text and the launch geometry it was captured on.
    A kernel source changed without a fresh capture fails here (and bench.py would report `frac: null`)."""
    from paper_2506_19866_b200 import build, inst_counts as IC
    build.build()
    from paper_2506_19866_b200 import binding as B
    counts = IC.load()
    for name in ("mtb", "hpg", "large", "paper_mtb", "paper_hpg"):
        c = counts[name]
        family, _ = IC.KERNELS[c["kernel"]]
        tree, lib = IC.tree_source_id(c["kernel"]), B.sa_kernel_source_id(family)
        assert lib == tree, f"libternary_sa.so carries another {c['kernel']} source than the tree: rebuild"
        assert c.get("source_id") == tree, (f"{name}: the instruction count was captured on kernel source {c.get('source_id')}, the tree has "
                                            f"{tree}: re-capture (python -m paper_2506_19866_b200.inst_counts update ...)")
        assert c["geometry"]["chains"] > 0 and c["geometry"]["threads_per_cta"] > 0
    # the check bench.py makes, on made-up handles
    c = counts["mtb"]
    launch = {k: v for k, v in c["geometry"].items() if k != "chains"}
    lib = B.sa_kernel_source_id(B.SA_KERNEL_DENSE)
    assert IC.stale_reason(c, "tsa_run_dense", lib, c["geometry"]["chains"], launch) is None
    assert "geometry" in IC.stale_reason(c, "tsa_run_dense", lib, c["geometry"]["chains"], dict(launch, chains_per_cta=16))
    assert "geometry" in IC.stale_reason(c, "tsa_run_dense", lib, 1024, launch)
    assert "source" in IC.stale_reason(c, "tsa_run_dense", "0" * 16, c["geometry"]["chains"], launch)
    assert "kernel" in IC.stale_reason(c, "tsa_run_static", lib, c["geometry"]["chains"], launch)
    with pytest.raises(B.SaError):
        B.sa_kernel_source_id(1)
