#!/usr/bin/env python
"""Benchmark of the SA hot path (BASELINE.json metric: SA chain-steps/s and node-updates/s on
one B200; % of the integer-issue roofline).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload mtb]

One bench "step" = one whole pass of the hot path over the workload: R fresh chains advanced
through the complete annealing schedule by ONE sa_run call (mtb: 4096 chains x 20 000 SA steps).
`value` times sa_run only (problem and chains resident in HBM); `e2e` times sa_create (host
buffers -> device) + sa_run + sa_best (device -> host) through the C ABI.  `--impl reference`
times the CPU oracle, as it stands, on a bounded sample of the same workload.  The paper's own model
(workloads paper_hpg / paper_mtb: sap_create / sap_run / sap_best) is measured the same way.
With --gpus N > 1 and no torchrun environment the script starts the N ranks itself.
"""
from __future__ import annotations

import argparse
import hashlib
import json
import os
import socket
import statistics
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

from paper_2506_19866_b200 import inst_counts as IC  # noqa: E402
from paper_2506_19866_b200 import problems as PB  # noqa: E402

METRIC = "sa_chain_steps_per_sec"
UNIT = "chain-steps/s"
WORKLOADS = sorted(PB.CONFIGS) + ["paper_hpg", "paper_mtb"]
# warp-instructions one chain-step executes, per kernel, from the committed ncu captures (smsp__inst_executed.sum
# of one launch / its chain-steps); bench.py multiplies them by the chain-steps/s it measures live


def _measured_peaks():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return json.load(f)
    except Exception:
        return {}


def _inst_counts():
    return IC.load()


def cpu_model() -> str:
    try:
        with open("/proc/cpuinfo") as f:
            for line in f:
                if line.lower().startswith("model name"):
                    return line.split(":", 1)[1].strip()
    except Exception:
        pass
    return "unknown"


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


def is_paper(name: str) -> bool:
    return name.startswith("paper_")


def _workload(name: str, args):
    spec = PB.PAPER_CONFIGS[name] if is_paper(name) else PB.CONFIGS[name]
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


def paper_bench_schedule(prob, chains, sa_steps, chain_id_base=0):
    """The paper's cooling (T = 1000, rho = 0.99) with steps_per_level = sa_steps: a bench
    step runs the first temperature level (the paper's n_iterations = 5000 at the default sa_steps);
    the table is as wide as the largest objective, so no worse move is rejected outright."""
    return PB.paper_schedule(chains, 8, sa_steps, prob.max_objective, chain_id_base=chain_id_base)


def self_launch(args) -> int:
    """python bench.py --gpus N without a torchrun environment: start the N ranks (one per GPU)."""
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    return subprocess.call(cmd)


# ------------------------------------------------------------------------------------ ours
def run_ours(args) -> dict:
    import torch
    from paper_2506_19866_b200 import binding as B

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py --impl ours needs a CUDA device (there is no CPU fallback)")
    if world != args.gpus:
        raise SystemExit(f"bench.py: --gpus {args.gpus} but WORLD_SIZE={world}")
    if torch.cuda.device_count() < max(args.gpus, local + 1):
        raise SystemExit(f"bench.py: --gpus {args.gpus} needs {args.gpus} visible CUDA devices, found {torch.cuda.device_count()}")
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

    def api(name):
        """(make problem, make schedule, create, run, best, destroy, fitness, info) of a workload's model."""
        if is_paper(name):
            prob = PB.make_paper_problem(name, B.sap_simulate)
            return (prob, lambda ch, st: paper_bench_schedule(prob, ch, st, rank_chain_base(rank, ch)),
                    lambda p, s: B.sap_create(p, s, B.SAP_CONSTRAINED), B.sap_run, B.sap_best, B.sap_destroy, B.sap_get_fitness,
                    lambda h: {"paper": B.sap_get_info(h)})
        prob = PB.make_problem(name, B.sa_simulate)
        return (prob, lambda ch, st: PB.make_schedule(ch, st, chain_id_base=rank_chain_base(rank, ch)),
                B.sa_create, B.sa_run, B.sa_best, B.sa_destroy, B.sa_get_fitness,
                lambda h: {"launch": B.sa_get_info(h), "dense": B.sa_get_dense_info(h)})

    def measure(name, chains, sa_steps, steps, warmup, want_e2e, want_cold=False):
        # inputs: synthetic, seeded; the ground-truth time courses come from the library's own
        # simulate call (the oracle is not on this path)
        prob, mk_sched, create, run, best_of, destroy, fitness, info_of = api(name)
        sched = mk_sched(chains, sa_steps)
        res = {"prob": prob, "sched": sched}
        if want_cold:
            # first handle of the process: NVRTC compile + host planner + first launch, never hidden by warm-up
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            h = create(prob, sched)
            t1 = time.perf_counter()
            run(h, 1)
            torch.cuda.synchronize()
            res["cold_start_ms"] = {"sa_create": (t1 - t0) * 1e3, "first_sa_run_1_step": (time.perf_counter() - t1) * 1e3}
            destroy(h)
        flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")   # > 126 MB L2
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
        info = best = None
        digests = []
        for it in range(warmup + steps):
            h = create(prob, sched)
            flush.fill_(it & 0xFF)
            if it == warmup:
                barrier()
            if it >= warmup:
                ev[it - warmup][0].record(stream)
            run(h, sa_steps)
            if it >= warmup:
                ev[it - warmup][1].record(stream)
            if it == warmup + steps - 1:
                barrier()
                info = info_of(h)
                best = best_of(h, prob.n_params)
            if it >= warmup:
                # determinism of the timing protocol: every repeat must end in the same state
                fc, fb = fitness(h, chains)
                digests.append(hashlib.sha1(fc.tobytes() + fb.tobytes()).hexdigest()[:16])
            destroy(h)
        ms = [a.elapsed_time(b) for a, b in ev]
        res.update({"ms": ms, "total_ms": max_over_ranks(sum(ms), dist), "info": info, "best": best,
                    "chain_steps": chains * sa_steps * steps * world, "repeats_identical": len(set(digests)) == 1,
                    "state_digest": digests[0]})
        if want_e2e:
            # end to end through the public API: host buffers in, best vector out, every step
            barrier()
            t0 = time.perf_counter()
            for it in range(steps):
                h = create(prob, sched)
                run(h, sa_steps)
                best = best_of(h, prob.n_params)
                destroy(h)
            barrier()
            dt = torch.tensor([time.perf_counter() - t0], dtype=torch.float64, device="cuda")
            if dist is not None:
                dist.all_reduce(dt, op=dist.ReduceOp.MAX)
            arrays = [prob.edge_src, prob.edge_dst, prob.init_state, sched.accept]
            arrays += [prob.fast, prob.ref] if is_paper(name) else [prob.th_lo, prob.th_hi, prob.obs_times, prob.clamp, prob.obs]
            res["e2e"] = {"value": chains * sa_steps * steps * world / float(dt.item()), "unit": UNIT,
                          "h2d_bytes_per_step": int(sum(np.asarray(a).nbytes for a in arrays)),
                          "d2h_bytes_per_step": int(prob.n_params + 8),
                          "plan": "warm: sa_create finds the host plans of this problem in its cache (every handle after the first)"}
            if not is_paper(name):
                # the same loop with the cache emptied before every create: each step also pays the host planner
                barrier()
                t0 = time.perf_counter()
                for it in range(steps):
                    B.sa_clear_plan_cache()
                    h = create(prob, sched)
                    run(h, sa_steps)
                    best = best_of(h, prob.n_params)
                    destroy(h)
                barrier()
                dt = torch.tensor([time.perf_counter() - t0], dtype=torch.float64, device="cuda")
                if dist is not None:
                    dist.all_reduce(dt, op=dist.ReduceOp.MAX)
                res["e2e"]["cold_plan"] = {"value": chains * sa_steps * steps * world / float(dt.item()), "unit": UNIT,
                                           "note": "sa_clear_plan_cache() before every sa_create: a first handle on a new problem"}
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

    def kernel_name(name, info):
        if is_paper(name):
            return "tsp_run"
        return {2: "run_kernel", 3: "run_warp_kernel", 4: "tsa_run_static", 5: "tsa_run_dense"}.get(info["launch"]["variant"], "?")

    def roofline(name, prob, chains, sa_steps, m, sms, sm_hz, imma):
        """Integer-issue roofline of the sa_run kernel: `frac` = issue slots used = executed warp-instructions
        per second / (SMs x 4 schedulers x f); `useful_frac` = algorithmic scalar operations per second /
        (SMs x 4 x 32 lanes x f), which extra instructions cannot inflate."""
        kernel_s = statistics.mean(m["ms"]) * 1e-3
        rate = chains * sa_steps / kernel_s                       # chain-steps/s of one launch on this rank
        issue_peak = sms * 4 * sm_hz
        kn = kernel_name(name, m["info"])
        cnt = _inst_counts().get(name, {})
        r = {"bound": "alu", "unit": "T warp-instr/s", "peak": issue_peak / 1e12,
             "peak_source": f"{sms} SMs x 4 schedulers x {sm_hz/1e6:.0f} MHz (MEASURED_PEAKS.json sm_max_mhz; DESIGN.md §7)",
             "kernel": kn, "kernel_ms": kernel_s * 1e3,
             # HBM traffic of the launch is the stage + write-back of the chains (2P + 8 bytes per chain each way,
             # ~6 MB per launch in profiles/r2d_mtb_dense.md); it is not re-measured in this run
             "traffic": None,
             "alg_ops_per_chain_step": prob.alg_ops_per_step,
             "useful_frac": prob.alg_ops_per_step * rate / (issue_peak * 32)}
        # a count only applies to the kernel text and launch geometry it was captured on (inst_counts.py)
        family = IC.KERNELS.get(kn, (None,))[0]
        stale = (IC.stale_reason(cnt, kn, B.sa_kernel_source_id(family), chains, m["info"].get("launch") or m["info"]["paper"]) if family
                 else f"no instruction count for kernel {kn} on workload {name} in profiles/inst_counts.json")
        if stale is None:
            r["warp_inst_per_chain_step"] = cnt["warp_inst_per_chain_step"]
            r["warp_inst_source"] = cnt.get("source")
            r["achieved"] = cnt["warp_inst_per_chain_step"] * rate / 1e12
            r["frac"] = cnt["warp_inst_per_chain_step"] * rate / issue_peak
            r["inst_per_node_update"] = cnt["warp_inst_per_chain_step"] / prob.node_updates_per_step
            if cnt.get("smem_wavefronts_per_chain_step"):
                # the gather kernels' ceiling is the shared-memory data pipe, one 128-byte wavefront per clock per SM
                r["shared_pipe"] = {"wavefronts_per_chain_step": cnt["smem_wavefronts_per_chain_step"],
                                    "source": cnt.get("smem_source"), "peak": "1 wavefront per clock per SM",
                                    "frac": cnt["smem_wavefronts_per_chain_step"] * rate / (sms * sm_hz)}
        else:
            r["achieved"] = None
            r["frac"] = None
            r["frac_note"] = stale
        if not is_paper(name) and m["info"]["launch"]["variant"] == 5 and imma:
            # second ceiling of the dense kernel: MMA instructions per time step against the rate of the
            # legacy tensor path measured in this run (sa_imma_peak)
            di = m["info"]["dense"]
            per_step = prob.n_steps * di["immas_per_step"]
            peak = imma["imma_sp_16864"] if di["sparse"] else imma["imma_16832"]
            r["tensor_pipe"] = {"imma_per_chain_step": per_step, "sparse_2of4": bool(di["sparse"]),
                                "achieved_imma_per_s": per_step * rate, "peak_imma_per_s": peak,
                                "peak_source": "sa_imma_peak, measured in this run", "frac": per_step * rate / peak}
            # On this tensor path an IMMA holds its sub-partition's issue port for its whole slot: the rate above is
            # one IMMA per 9 clocks per scheduler and nothing else issues meanwhile (measured: profiles/r2c_microbench.md,
            # DESIGN.md §7).  Scheduler clocks accounted for = IMMA slots + one clock per other warp-instruction.
            if r.get("warp_inst_per_chain_step"):
                imma_clk = issue_peak / peak
                clocks = per_step * imma_clk + (r["warp_inst_per_chain_step"] - per_step)
                r["exclusive_issue"] = {"clocks_per_imma": imma_clk, "scheduler_clocks_per_chain_step": clocks,
                                        "frac": clocks * rate / issue_peak,
                                        "note": "fraction of scheduler clocks that hold an IMMA slot or issue another instruction"}
        return r

    name = args.workload
    spec, chains, sa_steps = _workload(name, args)
    sampler = ClockSampler(local).start() if rank == 0 else None
    main = measure(name, chains, sa_steps, args.steps, args.warmup, True, want_cold=True)
    clocks = sampler.stop() if sampler else None
    prob = main["prob"]
    value = main["chain_steps"] / (main["total_ms"] * 1e-3)

    out = None
    if rank == 0:
        peaks = _measured_peaks()
        sm_hz = float(peaks.get("sm_max_mhz", 1965.0)) * 1e6
        sms = torch.cuda.get_device_properties(local).multi_processor_count
        imma = None
        if not is_paper(name):
            try:
                imma = B.sa_imma_peak()
            except Exception:
                imma = None
        dtype = ("int8 (byte-lane tables: PRMT look-up, integer adds and compares)" if is_paper(name)
                 else "int8 (mma.sync s8 x s8 -> s32, byte-lane SWAR thresholds)")
        out = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": main["total_ms"] / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": dtype, "data": "synthetic",
            "config": {"workload": (f"{name}: paper model N={prob.n_nodes} E={prob.n_edges} ({prob.n_params} parameters) K={prob.n_cond} "
                                    f"T={prob.n_steps}, constraints on, R={chains} chains/GPU x {sa_steps} SA steps" if is_paper(name) else
                                    f"{name}-shaped: N={prob.n_nodes} E={prob.n_edges} K={prob.n_cond} "
                                    f"T={prob.n_steps} n_obs={prob.n_obs}, R={chains} chains/GPU x {sa_steps} SA steps"),
                       "chains_per_gpu": chains, "sa_steps": sa_steps, "seed": prob.seed, "sa_seed": PB.SA_SEED,
                       "l2": "256 MiB buffer written between timed steps",
                       "parallelism": "chain-range partition, no collective" if world > 1 else "single GPU",
                       **main["info"]},
            "node_updates_per_sec": value * prob.node_updates_per_step,
            "best_fitness": int(main["best"][0]), "ground_truth_fitness": int(prob.n_flipped) if not is_paper(name) else None,
            "repeats_identical": main["repeats_identical"], "state_digest": main["state_digest"],
            "cold_start_ms": main.get("cold_start_ms"),
            "gpu_launches": args.steps,
            "e2e": main["e2e"], "clocks": clocks,
            "roofline": roofline(name, prob, chains, sa_steps, main, sms, sm_hz, imma),
        }
        if world == 1 and not args.no_extra:
            try:
                pk = B.sa_int32_peak()
                out["roofline"]["measured_issue_rates_warp_instr_per_s"] = {k: pk[k] for k in ("iadd3", "lop3", "imad", "mixed")}
                out["roofline"]["measured_sm_hz"] = pk["sm_hz"]
                if out["roofline"].get("achieved"):
                    out["roofline"]["frac_of_measured_iadd3_rate"] = out["roofline"]["achieved"] * 1e12 / pk["iadd3"]
            except Exception as e:  # pragma: no cover
                out["roofline"]["measured_issue_rates_error"] = str(e)
            extra = {}
            jobs = []
            if name == "mtb":
                jobs = [("hpg", None, None), ("large", None, None)]
                jobs += [("mtb", r, PB.SCALING_STEPS) for r in PB.SCALING_CHAINS]
                # the paper's own model at three of its thread counts (Table 2): one chain per thread there
                jobs += [("paper_mtb", 1024, 5000), ("paper_mtb", 10240, 5000), ("paper_mtb", 102400, 500), ("paper_hpg", 10240, 5000)]
            for wn, r, s in jobs:
                sp = PB.PAPER_CONFIGS[wn] if is_paper(wn) else PB.CONFIGS[wn]
                r, s = r or sp.n_chains, s or sp.sa_steps
                m = measure(wn, r, s, 2, 1, False)
                v = m["chain_steps"] / (m["total_ms"] * 1e-3)
                key = wn if (r, s) == (sp.n_chains, sp.sa_steps) else f"{wn}_R{r}_S{s}"
                rf = roofline(wn, m["prob"], r, s, m, sms, sm_hz, imma)
                extra[key] = {"value": v, "unit": UNIT, "node_updates_per_sec": v * m["prob"].node_updates_per_step,
                              "roofline_frac": rf["frac"], "useful_frac": rf["useful_frac"], "kernel": rf["kernel"],
                              **({"exclusive_issue_frac": rf["exclusive_issue"]["frac"]} if "exclusive_issue" in rf else {}),
                              **({"shared_pipe_frac": rf["shared_pipe"]["frac"]} if "shared_pipe" in rf else {}),
                              "ms_per_step": m["total_ms"] / 2, "repeats_identical": m["repeats_identical"], **m["info"]}
            if name == "mtb":
                # the paper's level structure (Table 1) with the synchronisation on the device
                extra["mtb_level_sync_all_chains"] = measure_levels(name, chains, sa_steps, 2, 1)
            out["other_workloads"] = extra
            out["cpu_baseline"] = cpu_baseline(name, prob)
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()
    return out


# ------------------------------------------------------------------------------------ oracle legs
def _oracle_for(prob):
    if is_paper(prob.name):
        from oracle import oracle_paper as OP
        return OP.PaperOracle(prob), {"constrained": True}
    from oracle import oracle as O
    return O.Oracle(prob), {}


def _oracle_sample(prob, chains, sa_steps, threads):
    orc, kw = _oracle_for(prob)
    if is_paper(prob.name):
        sched = paper_bench_schedule(prob, max(chains, 1), PB.PAPER_CONFIGS[prob.name].sa_steps)
    else:
        sched = PB.make_schedule(max(chains, 1), PB.CONFIGS[prob.name].sa_steps if prob.name in PB.CONFIGS else sa_steps)
    t0 = time.perf_counter()
    orc.run_chains(sched, range(chains), sa_steps, threads=threads, trace=False, **kw)
    return chains * sa_steps / (time.perf_counter() - t0)


_ORACLE_S_PER_STEP = {"tiny": 1.5e-5, "hpg": 3e-5, "mtb": 4e-4, "large": 1.1e-2, "paper_hpg": 7e-6, "paper_mtb": 3e-5}


def cpu_baseline(name: str, prob) -> dict:
    """The oracle as it stands on this box's host cores, bounded sample (about 10-30 s of CPU work):
    the single-threaded program, and the same program replicated over independent chains on every core."""
    cores = os.cpu_count() or 1
    per_step_s = _ORACLE_S_PER_STEP.get(name, 4e-4)
    chains = 2 * cores
    sa_steps = max(10, int(12.0 / per_step_s / chains))
    v = _oracle_sample(prob, chains, sa_steps, cores)
    one_steps = max(10, int(4.0 / per_step_s))
    v1 = _oracle_sample(prob, 1, one_steps, 1)
    return {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "cpu": cpu_model(),
            "single_thread": {"value": v1, "unit": UNIT, "sample": f"1 chain x {one_steps} SA steps"},
            "sample": f"{chains} chains x {sa_steps} SA steps of the {name} workload, "
                      f"single-threaded oracle code replicated over {cores} host threads"}


def run_reference(args) -> dict:
    """--impl reference: the CPU oracle on the same config, metric and unit (rank 0 only)."""
    if int(os.environ.get("RANK", "0")) != 0:
        return None
    name = args.workload
    spec, chains, sa_steps = _workload(name, args)
    if is_paper(name):
        from oracle import oracle_paper as OP
        prob = PB.make_paper_problem(name, OP.simulate_fn)
        shape = f"{name}: paper model N={prob.n_nodes} E={prob.n_edges} K={prob.n_cond} T={prob.n_steps}, constraints on"
    else:
        from oracle import oracle as O
        prob = PB.make_problem(name, O.simulate_fn)
        shape = f"{name}-shaped: N={prob.n_nodes} E={prob.n_edges} K={prob.n_cond} T={prob.n_steps} n_obs={prob.n_obs}"
    cores = os.cpu_count() or 1
    per_step_s = _ORACLE_S_PER_STEP.get(name, 4e-4)
    s_chains = cores
    s_steps = max(5, int(2.0 / per_step_s / s_chains))              # ~2 s of CPU work per bench step
    for _ in range(args.warmup):
        _oracle_sample(prob, s_chains, max(5, s_steps // 4), cores)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        _oracle_sample(prob, s_chains, s_steps, cores)
    dt = time.perf_counter() - t0
    v = s_chains * s_steps * args.steps / dt
    sample = (f"each step = {s_chains} chains x {s_steps} SA steps of the {name} workload "
              f"(full config: {chains} chains x {sa_steps}), oracle replicated over {cores} host threads")
    return {"impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": dt / args.steps * 1e3, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "int (byte per state)", "data": "synthetic",
            "config": {"workload": f"{shape}, R={chains} chains x {sa_steps} SA steps", "sample": sample},
            "node_updates_per_sec": v * prob.node_updates_per_step,
            "cpu_baseline": {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "cpu": cpu_model(), "sample": sample},
            "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", choices=["ours", "reference"], default="ours")
    ap.add_argument("--workload", choices=WORKLOADS, default="mtb")
    ap.add_argument("--chains", type=int, default=0, help="chains per GPU (default: the config's R)")
    ap.add_argument("--sa-steps", type=int, default=0, help="SA steps per bench step (default: the config's)")
    ap.add_argument("--no-extra", action="store_true", help="skip the other workloads, peak microbenchmark and cpu baseline")
    args = ap.parse_args()
    if args.gpus < 1:
        raise SystemExit("bench.py: --gpus must be >= 1")
    if args.impl == "ours" and args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        sys.exit(self_launch(args))
    out = run_reference(args) if args.impl == "reference" else run_ours(args)
    if out is not None:
        print(json.dumps(out))


if __name__ == "__main__":
    main()
