#!/usr/bin/env python
"""Benchmark of the SA hot path (BASELINE.json metric: SA chain-steps/s and node-updates/s on
one B200; % of the integer-issue roofline).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload mtb]

One bench "step" = one whole pass of the hot path over the workload: R fresh chains advanced
through the complete annealing schedule by ONE sa_run call (mtb: 4096 chains x 20 000 SA steps).
`value` times sa_run only (problem and chains resident in HBM); `e2e` times sa_create (host
buffers -> device) + sa_run + sa_best (device -> host) through the C ABI.  `--impl reference`
times the CPU oracle, as it stands, on a bounded sample of the same workload.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

from paper_2506_19866_b200 import problems as PB  # noqa: E402

METRIC = "sa_chain_steps_per_sec"
UNIT = "chain-steps/s"


def _measured_peaks():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return json.load(f)
    except Exception:
        return {}


class ClockSampler:
    """Samples SM clock and throttle reasons during the timed region (NVML, 100 ms period)."""

    def __init__(self, index: int):
        self.index, self.samples, self.reasons, self.max_mhz = index, [], set(), None
        self._stop = threading.Event()
        self._thr = None

    def start(self):
        try:
            import pynvml
            pynvml.nvmlInit()
            self._nv = pynvml
            self._dev = pynvml.nvmlDeviceGetHandleByIndex(self.index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self._dev, pynvml.NVML_CLOCK_SM)
        except Exception:
            self._nv = None
            return self
        self._thr = threading.Thread(target=self._loop, daemon=True)
        self._thr.start()
        return self

    def _loop(self):
        nv = self._nv
        names = {
            getattr(nv, "nvmlClocksEventReasonHwSlowdown", 0x8): "hw_slowdown",
            getattr(nv, "nvmlClocksEventReasonHwThermalSlowdown", 0x40): "hw_thermal_slowdown",
            getattr(nv, "nvmlClocksEventReasonSwThermalSlowdown", 0x20): "sw_thermal_slowdown",
            getattr(nv, "nvmlClocksEventReasonSwPowerCap", 0x4): "sw_power_cap",
        }
        while not self._stop.is_set():
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self._dev, nv.NVML_CLOCK_SM))
                try:
                    mask = nv.nvmlDeviceGetCurrentClocksEventReasons(self._dev)
                except Exception:
                    mask = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self._dev)
                for bit, name in names.items():
                    if mask & bit:
                        self.reasons.add(name)
            except Exception:
                pass
            self._stop.wait(0.1)

    def stop(self) -> dict:
        self._stop.set()
        if self._thr:
            self._thr.join(timeout=2)
        return {"sm_mhz": statistics.median(self.samples) if self.samples else None,
                "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons), "samples": len(self.samples)}


def _workload(name: str, args):
    spec = PB.CONFIGS[name]
    chains = args.chains or spec.n_chains
    sa_steps = args.sa_steps or spec.sa_steps
    return spec, chains, sa_steps


def rank_chain_base(rank: int, chains_per_gpu: int) -> int:
    """Chain-range partition: rank r owns global chains [r*R, (r+1)*R) (reading 25)."""
    return rank * chains_per_gpu


def max_over_ranks(ms: float, dist, device="cuda") -> float:
    """Device time of the slowest rank (the job's time); dist = torch.distributed or None."""
    import torch
    t = torch.tensor([ms], dtype=torch.float64, device=device)
    if dist is not None:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


# ------------------------------------------------------------------------------------ ours
def run_ours(args) -> dict:
    import torch
    from paper_2506_19866_b200 import binding as B

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py --impl ours needs a CUDA device (there is no CPU fallback)")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    B.use_torch_plumbing()
    stream = torch.cuda.current_stream()

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    def measure(name, chains, sa_steps, steps, warmup, want_e2e):
        # inputs: synthetic, seeded; the ground-truth time courses come from the library's own
        # sa_simulate (the oracle is not on this path)
        prob = PB.make_problem(name, B.sa_simulate)
        sched = PB.make_schedule(chains, sa_steps, chain_id_base=rank_chain_base(rank, chains))
        flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")   # > 126 MB L2
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
        info = None
        best = None
        dense = None
        for it in range(warmup + steps):
            h = B.sa_create(prob, sched)
            flush.fill_(it & 0xFF)
            if it == warmup:
                barrier()
            if it >= warmup:
                ev[it - warmup][0].record(stream)
            B.sa_run(h, sa_steps)
            if it >= warmup:
                ev[it - warmup][1].record(stream)
            if it == warmup + steps - 1:
                barrier()
                info = B.sa_get_info(h)
                dense = B.sa_get_dense_info(h)
                best = B.sa_best(h, prob.n_params)
            B.sa_destroy(h)
        ms = [a.elapsed_time(b) for a, b in ev]
        kernel_ms = sum(ms)
        total_ms = max_over_ranks(kernel_ms, dist)
        res = {"prob": prob, "sched": sched, "ms": ms, "total_ms": total_ms, "info": info, "best": best, "dense": dense,
               "chain_steps": chains * sa_steps * steps * world}
        if want_e2e:
            # end to end through the public API: host buffers in, best vector out, every step
            barrier()
            t0 = time.perf_counter()
            for it in range(steps):
                h = B.sa_create(prob, sched)
                B.sa_run(h, sa_steps)
                best = B.sa_best(h, prob.n_params)
                B.sa_destroy(h)
            barrier()
            dt = torch.tensor([time.perf_counter() - t0], dtype=torch.float64, device="cuda")
            if dist is not None:
                dist.all_reduce(dt, op=dist.ReduceOp.MAX)
            h2d = sum(np.asarray(a).nbytes for a in (prob.edge_src, prob.edge_dst, prob.th_lo, prob.th_hi,
                                                    prob.obs_times, prob.init_state, prob.clamp, prob.obs,
                                                    sched.accept))
            res["e2e"] = {"value": chains * sa_steps * steps * world / float(dt.item()), "unit": UNIT,
                          "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(prob.n_params + 8)}
        return res

    def measure_levels(name, chains, sa_steps, steps, warmup, group=0):
        prob = PB.make_problem(name, B.sa_simulate)
        sched = PB.make_schedule(chains, sa_steps, chain_id_base=rank_chain_base(rank, chains))
        n_levels = sa_steps // sched.steps_per_level
        ms = []
        for it in range(warmup + steps):
            h = B.sa_create(prob, sched)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            torch.cuda.synchronize()
            e0.record(stream)
            B.sa_run_levels(h, n_levels, group)
            e1.record(stream)
            torch.cuda.synchronize()
            if it >= warmup:
                ms.append(e0.elapsed_time(e1))
            best = B.sa_best(h, prob.n_params)
            B.sa_destroy(h)
        v = chains * sa_steps * len(ms) / (sum(ms) * 1e-3)
        return {"value": v, "unit": UNIT, "levels": n_levels, "steps_per_level": sched.steps_per_level, "group_size": group or chains,
                "ms_per_step": sum(ms) / len(ms), "best_fitness": int(best[0]),
                "kernels_per_level": "sa_run kernel + group_argmin_kernel + level_broadcast_kernel"}

    name = args.workload
    spec, chains, sa_steps = _workload(name, args)
    sampler = ClockSampler(local).start() if rank == 0 else None
    main = measure(name, chains, sa_steps, args.steps, args.warmup, True)
    clocks = sampler.stop() if sampler else None
    prob = main["prob"]
    value = main["chain_steps"] / (main["total_ms"] * 1e-3)

    out = None
    if rank == 0:
        peaks = _measured_peaks()
        sm_max_hz = float(peaks.get("sm_max_mhz", 1965.0)) * 1e6
        sms = main["info"]["sm_count"]
        issue_peak = sms * 4 * 32 * sm_max_hz                      # lane-ops/s: 4 schedulers x 32 lanes per SM-clock
        kernel_s = statistics.mean(main["ms"]) * 1e-3
        alg_ops = prob.alg_ops_per_step * chains * sa_steps       # per launch (one rank)
        achieved = alg_ops / kernel_s
        out = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": main["total_ms"] / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "int8 (mma.sync s8 x s8 -> s32, byte-lane SWAR thresholds)", "data": "synthetic",
            "config": {"workload": f"{name}-shaped: N={prob.n_nodes} E={prob.n_edges} K={prob.n_cond} "
                                   f"T={prob.n_steps} n_obs={prob.n_obs}, R={chains} chains/GPU x {sa_steps} SA steps",
                       "chains_per_gpu": chains, "sa_steps": sa_steps, "seed": prob.seed, "sa_seed": PB.SA_SEED,
                       "l2": "256 MiB buffer written between timed steps",
                       "parallelism": "chain-range partition, no collective" if world > 1 else "single GPU",
                       "launch": main["info"]},
            "node_updates_per_sec": value * prob.node_updates_per_step,
            "best_fitness": int(main["best"][0]), "ground_truth_fitness": int(prob.n_flipped),
            "gpu_launches": args.steps,
            "e2e": main["e2e"], "clocks": clocks,
            "roofline": {"bound": "alu", "achieved": achieved / 1e12, "peak": issue_peak / 1e12,
                         "unit": "T int-lane-op/s", "frac": achieved / issue_peak,
                         # dram__bytes_read.sum + dram__bytes_write.sum of one sa_run launch, from the ncu capture in
                         # profiles/r1_v6_run_dense_sparse_unrolled.md (stage + write back of the chains; HBM is not the bound)
                         "traffic": 6.10e6 if name == "mtb" else None,
                         "peak_source": f"{sms} SMs x 4 schedulers x 32 lanes x {sm_max_hz/1e6:.0f} MHz "
                                        "(MEASURED_PEAKS.json sm_max_mhz; DESIGN.md §7)",
                         "alg_ops_per_chain_step": prob.alg_ops_per_step},
        }
        if main["info"]["variant"] == 5:
            # second ceiling of the dense kernel: MT*KS IMMA.16832.S8 per time step against the measured
            # 0.5 IMMA per clock per SM of the legacy tensor path on B200
            di = main["dense"]
            per_step = prob.n_steps * di["row_tiles"] * (di["col_steps"] // 2 if di["sparse"] else di["col_steps"])
            rate = 0.443 if di["sparse"] else 0.5     # measured: IMMA.SP.16864 / IMMA.16832 per clock per SM
            immas = per_step * chains * sa_steps / kernel_s
            out["roofline"]["tensor_pipe"] = {"imma_per_chain_step": per_step, "sparse_2of4": bool(di["sparse"]),
                                              "achieved_imma_per_s": immas, "peak_imma_per_s": rate * sms * sm_max_hz,
                                              "frac": immas / (rate * sms * sm_max_hz)}
            out["config"]["dense"] = di
        if world == 1 and not args.no_extra:
            try:
                pk = B.sa_int32_peak()
                out["roofline"]["measured_issue_rates_warp_instr_per_s"] = {k: pk[k] for k in ("iadd3", "lop3", "imad", "mixed")}
                out["roofline"]["measured_sm_hz"] = pk["sm_hz"]
                out["roofline"]["frac_of_measured_mixed"] = achieved / (pk["mixed"] * 32)
            except Exception as e:  # pragma: no cover
                out["roofline"]["measured_issue_rates_error"] = str(e)
            extra = {}
            jobs = [("hpg", None, None), ("large", None, None)] if name == "mtb" else []
            jobs += [("mtb", r, PB.SCALING_STEPS) for r in PB.SCALING_CHAINS] if name == "mtb" else []
            for wn, r, s in jobs:
                sp = PB.CONFIGS[wn]
                r, s = r or sp.n_chains, s or sp.sa_steps
                m = measure(wn, r, s, 2, 1, False)
                v = m["chain_steps"] / (m["total_ms"] * 1e-3)
                key = wn if (r, s) == (sp.n_chains, sp.sa_steps) else f"{wn}_R{r}_S{s}"
                extra[key] = {"value": v, "unit": UNIT, "node_updates_per_sec": v * m["prob"].node_updates_per_step,
                              "roofline_frac": m["prob"].alg_ops_per_step * v / issue_peak,
                              "ms_per_step": m["total_ms"] / 2, "launch": m["info"]}
            if name == "mtb":
                # the paper's level structure (Table 1) with the synchronisation on the device
                lv = measure_levels(name, chains, sa_steps, 2, 1)
                extra["mtb_level_sync_all_chains"] = lv
            out["other_workloads"] = extra
            out["cpu_baseline"] = cpu_baseline(name, prob)
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()
    return out


# ------------------------------------------------------------------------------------ oracle legs
def _oracle_sample(prob, chains, sa_steps, threads):
    from oracle import oracle as O
    orc = O.Oracle(prob)
    sched = PB.make_schedule(max(chains, 1), PB.CONFIGS[prob.name].sa_steps if prob.name in PB.CONFIGS else sa_steps)
    t0 = time.perf_counter()
    orc.run_chains(sched, range(chains), sa_steps, threads=threads, trace=False)
    return chains * sa_steps / (time.perf_counter() - t0)


def cpu_baseline(name: str, prob) -> dict:
    """The oracle as it stands on this box's host cores, bounded sample (about 10-30 s of CPU work)."""
    cores = os.cpu_count() or 1
    per_step_s = {"tiny": 1.5e-5, "hpg": 3e-5, "mtb": 4e-4, "large": 1.1e-2}.get(name, 4e-4)
    chains = 2 * cores
    sa_steps = max(10, int(15.0 / per_step_s / chains))
    v = _oracle_sample(prob, chains, sa_steps, cores)
    return {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": f"{chains} chains x {sa_steps} SA steps of the {name}-shaped workload, "
                      f"single-threaded oracle code replicated over {cores} host threads"}


def run_reference(args) -> dict:
    """--impl reference: the CPU oracle on the same config, metric and unit (rank 0 only)."""
    if int(os.environ.get("RANK", "0")) != 0:
        return None
    from oracle import oracle as O
    name = args.workload
    spec, chains, sa_steps = _workload(name, args)
    prob = PB.make_problem(name, O.simulate_fn)
    cores = os.cpu_count() or 1
    per_step_s = {"tiny": 1.5e-5, "hpg": 3e-5, "mtb": 4e-4, "large": 1.1e-2}.get(name, 4e-4)
    s_chains = cores
    s_steps = max(5, int(2.0 / per_step_s / s_chains))              # ~2 s of CPU work per bench step
    for _ in range(args.warmup):
        _oracle_sample(prob, s_chains, max(5, s_steps // 4), cores)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        _oracle_sample(prob, s_chains, s_steps, cores)
    dt = time.perf_counter() - t0
    v = s_chains * s_steps * args.steps / dt
    sample = (f"each step = {s_chains} chains x {s_steps} SA steps of the {name}-shaped workload "
              f"(full config: {chains} chains x {sa_steps}), oracle replicated over {cores} host threads")
    return {"impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": dt / args.steps * 1e3, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "int (byte per state)", "data": "synthetic",
            "config": {"workload": f"{name}-shaped: N={prob.n_nodes} E={prob.n_edges} K={prob.n_cond} T={prob.n_steps} "
                                   f"n_obs={prob.n_obs}, R={chains} chains x {sa_steps} SA steps", "sample": sample},
            "node_updates_per_sec": v * prob.node_updates_per_step,
            "cpu_baseline": {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", choices=["ours", "reference"], default="ours")
    ap.add_argument("--workload", choices=sorted(PB.CONFIGS), default="mtb")
    ap.add_argument("--chains", type=int, default=0, help="chains per GPU (default: the config's R)")
    ap.add_argument("--sa-steps", type=int, default=0, help="SA steps per bench step (default: the config's)")
    ap.add_argument("--no-extra", action="store_true", help="skip the other workloads, peak microbenchmark and cpu baseline")
    args = ap.parse_args()
    out = run_reference(args) if args.impl == "reference" else run_ours(args)
    if out is not None:
        print(json.dumps(out))


if __name__ == "__main__":
    main()
