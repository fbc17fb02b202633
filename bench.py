#!/usr/bin/env python
"""Benchmark of the nuclear-pasta MD hot path (BASELINE.json metric: MD steps/s and pair interactions/s
at 409 600 nucleons; fraction of the B200 FP32/SFU roofline).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 4|2]

One "step" = one full MD step (first half kick + drift + box scaling + wrap, cell-list build, pair
force + energy, second half kick + KE + thermostat) of BASELINE config 4 (409 600 nucleons, Y_P = 0.30,
n = 0.08 fm^-3, T = 0.5 MeV, r_c = 20 fm, rescale every 10 steps) on seeded synthetic input.  The metric
names two sizes: the same line carries a `config2` block with the 51 200-nucleon numbers (BASELINE config 2),
measured in the same process after the config-4 legs.  By default --gpus N runs N independent replicas, one
process per GPU, and reports their aggregate ("replicas only"); --shard runs ONE simulation
with the targets of every force evaluation split over the ranks instead (never measured on
hardware: no multi-GPU node was available).  Prints ONE JSON line on rank 0.
"""
import argparse
import json
import math
import os
import statistics
import subprocess
import sys
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from paper_1412_8502_b200 import inputs  # noqa: E402

SM_COUNT = 148
FP32_LANES_PER_SM = 128  # 4 SMSPs x 32 lanes, one warp instruction per SMSP per clock
MUFU_LANES_PER_SM = 16


def peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    sm_max_mhz, hbm, src = 1965.0, 6650.0, "fallback (B200_PROFILING.md)"
    if os.path.exists(path):
        try:
            m = json.load(open(path))
            sm_max_mhz, hbm, src = float(m.get("sm_max_mhz", sm_max_mhz)), float(m.get("hbm_gbs", hbm)), "MEASURED_PEAKS.json"
        except Exception:
            pass
    return sm_max_mhz, hbm, src


def ncu_traffic(cfg):
    """roofline.traffic: dram__bytes_read.sum + dram__bytes_write.sum of ONE launch of the pair kernel, read from the
    committed `ncu --set full` summary of this round (profiles/), never a literal in this file.  (bytes, source) or
    (None, reason)."""
    import re

    unit = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9}
    for name in ("r3_k2_ncu_cfg%d.md" % cfg, "r2_k2_ncu_cfg%d.md" % cfg):  # the newest capture of the shipped kernel first
        path = os.path.join(ROOT, "profiles", name)
        if not os.path.exists(path):
            continue
        total, found = 0.0, 0
        for line in open(path):
            m = re.match(r"\|\s*`dram__bytes_(read|write)\.sum`\s*\|\s*([0-9.]+)\s*(\w+)", line)
            if m and m.group(3) in unit:
                total += float(m.group(2)) * unit[m.group(3)]
                found += 1
        if found == 2:
            return total, "profiles/" + name
    return None, "no committed ncu --set full summary for config %d" % cfg


def algorithmic_cost(Y_P):
    """FP32 lane-instructions and MUFU ops per ordered in-range pair:
    17 + 1 for a nuclear-only pair, +8 and +2 for a proton-proton pair (fraction Y_P^2 when uniform)."""
    fpp = Y_P * Y_P
    return 17.0 + 8.0 * fpp, 1.0 + 2.0 * fpp


class ClockSampler:
    """nvidia-smi clocks + throttle reasons sampled during the timed region (B200_PROFILING.md)."""

    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.proc = None
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except Exception:
            self.proc = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.proc is None:
            return out
        time.sleep(0.15)
        self.proc.terminate()
        try:
            text = self.proc.communicate(timeout=5)[0]
        except Exception:
            self.proc.kill()
            text = ""
        sm, mx, reasons = [], [], set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for line in text.splitlines():
            f = [t.strip() for t in line.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0]))
                mx.append(float(f[1]))
            except ValueError:
                continue
            for name, val in zip(names, f[3:7]):
                if val.lower().startswith("active"):
                    reasons.add(name)
        if sm:
            out.update(sm_mhz=statistics.median(sm), sm_max_mhz=max(mx), reasons=sorted(reasons), samples=len(sm))
        return out


def cpu_baseline(cfg, budget_s, seed=1, state=None, all_pairs=True):
    """The oracle as it stands, timed on the host cores.

    `value`: the oracle's own cell-list variant (orc_forces_cells: the same FP64 definition evaluated through the
    27 cells of width >= r_c, pinned against the all-pairs loop by P7) -- ONE FULL force + energy evaluation of the
    workload = one MD step (the O(N) integrator update is not in it; the force calculation is "by far
    the most time consuming part of each time step").  The paper's CPU code was list-based too.
    `all_pairs_extrapolated`: the O(N^2) definition itself on a bounded sample of targets against ALL N sources,
    scaled by N / n_sample -- kept beside it, labelled as the extrapolation it is."""
    import numpy as np

    import oracle

    c = inputs.CONFIGS[cfg]
    x, v, is_p, L = state if state is not None else inputs.config_state(cfg, seed)
    p = oracle.Params(r_c=c["r_c"])
    cores = oracle.num_threads()
    t0 = time.perf_counter()
    _, _, pe_fp64, npairs = oracle.forces_cells(x, is_p, L, p)
    dt = time.perf_counter() - t0
    out = {
        "value": 1.0 / dt, "unit": "steps/s", "cores": cores, "kind": "oracle",
        "sample": "one full FP64 force+energy evaluation of all %d targets through the oracle's 27-cell list "
                  "(orc_forces_cells) in %.2f s; not extrapolated%s" % (
                      c["N"], dt, "; on the state read back from the GPU run after its timed steps" if state is not None else ""),
        "ordered_pairs_per_s": npairs / dt, "PE_MeV": pe_fp64,
    }
    if all_pairs:
        rng = np.random.default_rng(0)
        probe = np.sort(rng.choice(c["N"], size=4 * cores, replace=False))
        t0 = time.perf_counter()
        oracle.forces(x, is_p, L, p, targets=probe)
        per_target = (time.perf_counter() - t0) / len(probe)
        n_sample = int(max(cores, min(c["N"], budget_s / max(per_target, 1e-9))))
        n_sample -= n_sample % cores
        sample = np.sort(rng.choice(c["N"], size=n_sample, replace=False))
        t0 = time.perf_counter()
        _, _, _, diag = oracle.forces(x, is_p, L, p, targets=sample)
        dt2 = time.perf_counter() - t0
        out["all_pairs_extrapolated"] = {
            "value": n_sample / (dt2 * c["N"]), "unit": "steps/s",
            "sample": "FP64 all-pairs forces+energy of %d of %d targets vs all %d sources in %.1f s, scaled by N/n_sample"
                      % (n_sample, c["N"], c["N"], dt2),
            "ordered_pairs_per_s": diag["ordered_pairs"] / dt2}
    return out


def run_reference(args, rank, world):
    """--impl reference: the oracle on the host cores, same metric/config.  A step = one full force+energy evaluation
    through the oracle's cell list (see cpu_baseline); the number of evaluations actually run is bounded so that the
    whole call ends within a few minutes, and stated."""
    if rank != 0:
        return
    state = inputs.config_state(args.config, 1)
    first = cpu_baseline(args.config, 0.0, state=state, all_pairs=False)
    t_eval = 1.0 / first["value"]
    total = max(1, args.steps + args.warmup)
    n_run = int(max(1, min(total, 150.0 / t_eval)))
    warm = min(args.warmup, n_run - 1)
    vals = []
    base = first
    for k in range(1, n_run):
        base = cpu_baseline(args.config, 0.0, state=state, all_pairs=False)
        if k >= warm:
            vals.append(base["value"])
    if not vals:
        vals = [first["value"]]
    for b_ in (first, base):  # (the state is the seeded start, not a GPU read-back)
        b_["sample"] = b_["sample"].replace("; on the state read back from the GPU run after its timed steps", "")
    v = len(vals) / sum(1.0 / a for a in vals)
    sample = base["sample"] + "; %d evaluations timed (%d asked for, bounded to ~150 s)" % (len(vals), args.steps)
    line = {
        "impl": "reference", "metric": "md_steps_per_s", "value": v, "unit": "steps/s", "n_gpus": args.gpus,
        # `steps` / `warmup` are what was really run and timed, so that steps x ms_per_step is this arm's timed region
        "steps": len(vals), "warmup": n_run - len(vals), "steps_asked": args.steps, "warmup_asked": args.warmup,
        "ms_per_step": 1e3 / v, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": workload_config(args.config, world),
        "cpu_baseline": {"value": v, "unit": "steps/s", "cores": base["cores"], "kind": "oracle", "sample": sample},
        "e2e": {"value": v, "unit": "steps/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }
    print(json.dumps(line), flush=True)


def workload_config(cfg, world, sharded=False):
    c = inputs.CONFIGS[cfg]
    return {
        "workload": "BASELINE config %d: %d nucleons, Y_P=%.2f, n=%.3f fm^-3, T=%.2f MeV, r_c=%g fm, dt=%g fm/c, "
                    "velocity rescale every %d steps, seeded uniform-random start" % (
                        cfg, c["N"], c["Y_P"], c["density"], c["T"], c["r_c"], c["dt"], c["thermostat_interval"]),
        "N": c["N"], "parallelism": ("one simulation, targets sharded over %d GPUs, force all-reduce (NCCL) per evaluation" % world)
        if sharded else "replicas x%d (one GPU each, no data-path collective)" % world,
        "l2": "flushed between timed steps (256 MB write); the 50 MB MD state is otherwise L2-resident by nature",
    }


def max_over_ranks(dev_s, e2e_s, dist, device="cuda"):
    """The contract's timing rule: every number is the MAX over ranks (replicas run independently)."""
    import torch

    t = torch.tensor([dev_s, e2e_s], dtype=torch.float64, device=device)
    if dist is not None:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return tuple(t.tolist())


def aggregate_rate(world, steps, seconds):
    """Whole-job steps/s of `world` independent replicas that each did `steps` steps in at most `seconds`."""
    return world * steps / seconds


def device_leg(sim, c, steps, warmup, flush, barrier, clock_gpu):
    """Device-resident timing of `steps` single MD steps, each bracketed by CUDA events on the simulation's stream (torch's
    current one), L2 flushed in between; then the same steps once more with the library's own event brackets around the
    kernel groups (K1 / K2 / K3) -- the brackets switch the captured-graph replay of a step off, so they are kept out of
    the headline region.  nvidia-smi clocks are sampled over both (clock_gpu = GPU index, None = do not sample)."""
    import torch

    for _ in range(max(warmup, 3)):
        sim.step(1, c["dt"])
    torch.cuda.synchronize()
    n0 = sim.launch_count()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    barrier()
    sampler = ClockSampler(clock_gpu) if clock_gpu is not None else None
    t_wall0 = time.perf_counter()
    for a, b in ev:
        flush.zero_()
        a.record()
        sim.step(1, c["dt"])
        b.record()
    barrier()
    t_wall = time.perf_counter() - t_wall0
    launches = sim.launch_count() - n0
    sim.set_timing(True)
    for _ in range(min(steps, 200)):
        flush.zero_()
        sim.step(1, c["dt"])
    barrier()
    clocks = sampler.stop() if sampler else None
    tm = sim.get_timing()
    sim.set_timing(False)
    per_step_ms = sorted(a.elapsed_time(b) for a, b in ev)
    pairs, pairs_nz = sim.pair_counts()  # ordered in-range pairs; those with a term that is not exactly 0 in FP32
    return {"wall_s": t_wall, "launches": launches, "clocks": clocks, "tm": tm, "per_step_ms": per_step_ms,
            "dev_s": sum(per_step_ms) * 1e-3, "pairs": pairs, "pairs_nz": pairs_nz}


def k2_roofline(c, pairs, pairs_nz, k2_s, fp32_peak):
    """(work-performed fraction, contract-formula fraction) of the FP32 peak for one pair-kernel launch of k2_s seconds."""
    c_fp32, _ = algorithmic_cost(c["Y_P"])
    return ((17.0 * pairs_nz + 8.0 * c["Y_P"] ** 2 * pairs) / k2_s / fp32_peak, pairs * c_fp32 / k2_s / fp32_peak)


def config2_block(args, flush, barrier, local_rank, fp32_peak):
    """The 51 200-nucleon half of the metric (BASELINE config 2; Fig. 1), measured like the headline."""
    import paper_1412_8502_b200 as pasta

    c = inputs.CONFIGS[2]
    prm = pasta.default_params(r_c=c["r_c"], thermostat_interval=c["thermostat_interval"], scale_per_step=c["scale_per_step"])
    with pasta.Sim(c["N"], c["Y_P"], c["density"], c["T"], params=prm, seed=args.seed) as sim:
        leg = device_leg(sim, c, args.steps, args.warmup, flush, barrier, local_rank)
        ke, pe = sim.energy()
    tm, n_ev = leg["tm"], max(1, leg["tm"]["force_evals"])
    k2_s = tm["force_ms"] * 1e-3 / n_ev
    frac, frac_contract = k2_roofline(c, leg["pairs"], leg["pairs_nz"], k2_s, fp32_peak)
    rate = args.steps / leg["dev_s"]
    return {"workload": workload_config(2, 1)["workload"], "N": c["N"], "md_steps_per_s": rate,
            "ms_per_step": 1e3 * leg["dev_s"] / args.steps, "steps": args.steps,
            "pair_interactions_per_s": {"unordered": 0.5 * leg["pairs"] * rate, "ordered": leg["pairs"] * rate,
                                        "ordered_pairs_per_step": leg["pairs"]},
            "kernel_ms": {"cells": tm["cells_ms"] / n_ev, "pair_force": 1e3 * k2_s, "integrate": tm["integrate_ms"] / n_ev},
            "roofline": {"bound": "alu", "kernel": "pair force (K2)", "frac": frac, "frac_contract_formula": frac_contract,
                         "peak": fp32_peak / 1e9, "unit": "G FP32 lane-instr/s", "nonzero_pairs_per_step": leg["pairs_nz"]},
            "gpu_launches": leg["launches"], "clocks": leg["clocks"], "energies_MeV": {"KE": ke, "PE": pe}}


def run_ours(args, rank, world, local_rank):
    import torch

    import paper_1412_8502_b200 as pasta

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist

        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    c = inputs.CONFIGS[args.config]
    N = c["N"]
    prm = pasta.default_params(r_c=c["r_c"], thermostat_interval=c["thermostat_interval"],
                               scale_per_step=c["scale_per_step"])
    for kv in filter(None, args.params.split(",")):  # pasta_params overrides, e.g. --params r_nuc=11.5,skip_exact_zeros=0
        key, val = kv.split("=")
        setattr(prm, key, type(getattr(prm, key))(float(val)))
    # replicas (default): rank r runs its own simulation (seed + r).  --shard: ONE simulation, replicated state, the
    # targets of every force evaluation split over the ranks and the partial forces summed with an NCCL all-reduce
    sharded = bool(args.shard) and world > 1
    sim = pasta.Sim(N, c["Y_P"], c["density"], c["T"], params=prm, seed=args.seed + (0 if sharded else rank))
    if sharded:
        sim.set_shard(rank, world)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    leg = device_leg(sim, c, args.steps, args.warmup, flush, barrier, local_rank if rank == 0 else None)
    t_wall, launches, clocks, tm, per_step_ms = leg["wall_s"], leg["launches"], leg["clocks"], leg["tm"], leg["per_step_ms"]
    dev_s, pairs, pairs_nz = leg["dev_s"], leg["pairs"], leg["pairs_nz"]
    ke, pe = sim.energy()

    # ---- end to end through the C ABI with HOST buffers: every step copies the state in and out ----
    # (a) serial chain: the host feeds every result back as the next input, so nothing can overlap
    hx, hv, hF = (torch.empty((N, 3), dtype=torch.float64).pin_memory() for _ in range(3))
    L, _ = sim.get_state_host(hx, hv, hF)
    e2e_steps = max(3, min(args.steps, 50))
    for _ in range(2):
        sim.set_state_host(hx, hv, None, hF, L)
        sim.step(1, c["dt"])
        L, _ = sim.get_state_host(hx, hv, hF)
    barrier()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        sim.set_state_host(hx, hv, None, hF, L)
        sim.step(1, c["dt"])
        L, _ = sim.get_state_host(hx, hv, hF)
    barrier()
    e2e_serial_s = time.perf_counter() - t0
    # (b) independent one-step requests (state in -> one MD step -> state out), pipelined by the library: uploads and
    # downloads run on side streams with double-buffered staging while the previous / next step is computed
    ins = [tuple(t.clone().pin_memory() for t in (hx, hv, hF)) for _ in range(2)]
    outs = [tuple(torch.empty((N, 3), dtype=torch.float64).pin_memory() for _ in range(3)) for _ in range(2)]

    def pipelined(n):
        for k in range(n):
            sim.set_state_host_async(*ins[k & 1], L=L)
            sim.step(1, c["dt"])
            sim.get_state_host_async(*outs[k & 1])
        sim.host_sync()

    pipelined(4)
    barrier()
    t0 = time.perf_counter()
    pipelined(e2e_steps)
    barrier()
    e2e_s = time.perf_counter() - t0
    e2e_serial_s = max_over_ranks(e2e_serial_s, 0.0, dist)[0]

    dev_s, e2e_s = max_over_ranks(dev_s, e2e_s, dist)
    if rank == 0:
        sm_max_mhz, hbm_gbs, peak_src = peaks()
        c_fp32, c_mufu = algorithmic_cost(c["Y_P"])
        k2_s = tm["force_ms"] * 1e-3 / max(1, tm["force_evals"])
        fp32_peak = SM_COUNT * FP32_LANES_PER_SM * sm_max_mhz * 1e6
        mufu_peak = SM_COUNT * MUFU_LANES_PER_SM * sm_max_mhz * 1e6
        # contract formula: every ordered pair with r < r_c is credited its algorithmic cost
        achieved_contract = pairs * c_fp32 / k2_s
        # work performed: only the pairs whose term is not exactly 0.0f in FP32 count (all pp pairs, np/nn pairs
        # inside the underflow distance) -- the headline `frac`
        achieved = (17.0 * pairs_nz + 8.0 * c["Y_P"] ** 2 * pairs) / k2_s
        traffic, traffic_src = ncu_traffic(args.config)
        roof_pairs = min(fp32_peak / c_fp32, mufu_peak / c_mufu)
        steps_per_s = aggregate_rate(1 if sharded else world, args.steps, dev_s)
        line = {
            "metric": "md_steps_per_s", "value": steps_per_s, "unit": "steps/s", "n_gpus": world,
            "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": 1e3 * dev_s / args.steps,
            "ms_per_step_stats": {"median": statistics.median(per_step_ms), "min": per_step_ms[0], "max": per_step_ms[-1]},
            "higher_is_better": True, "scaling": "strong" if sharded else "weak", "vs_baseline": None, "dtype": "f32",
            "data": "synthetic", "config": workload_config(args.config, world, sharded),
            "pair_interactions_per_s": {"unordered": 0.5 * pairs * steps_per_s, "ordered": pairs * steps_per_s,
                                        "ordered_pairs_per_step": pairs},
            # K1 and K3 move 76 and 192 algorithmic bytes per particle and step; they are
            # L2-resident and launch-latency-bound, so these are far below the HBM peak by construction
            "k1_k3_gbs": {"cells": 76.0 * N / (tm["cells_ms"] / max(1, tm["force_evals"]) * 1e-3) / 1e9,
                          "integrate": 192.0 * N / (tm["integrate_ms"] / max(1, tm["force_evals"]) * 1e-3) / 1e9,
                          "hbm_peak": hbm_gbs},
            "kernel_ms": {"cells": tm["cells_ms"] / max(1, tm["force_evals"]), "pair_force": 1e3 * k2_s,
                          "integrate": tm["integrate_ms"] / max(1, tm["force_evals"])},
            "roofline": {
                "bound": "alu", "kernel": "pair force (K2)", "achieved": achieved / 1e9, "peak": fp32_peak / 1e9,
                "unit": "G FP32 lane-instr/s, work performed: 17 per ordered in-range pair whose term is not exactly 0.0f "
                        "in FP32 + 8 per proton-proton pair (the pairs skip_exact_zeros never touches earn nothing)",
                "frac": achieved / fp32_peak,
                "frac_contract_formula": achieved_contract / fp32_peak,
                "contract_formula": "every ordered pair with r < r_c x %.2f FP32 (SURVEY 8(d)); algorithmic credit, "
                                    "not pipe utilisation" % c_fp32,
                "nonzero_pairs_per_step": pairs_nz, "skip_exact_zeros": int(prm.skip_exact_zeros),
                "frac_of_pair_roofline": (pairs / k2_s) / roof_pairs,
                "ordered_pairs_per_s": pairs / k2_s, "mufu_frac": (pairs * c_mufu / k2_s) / mufu_peak,
                "peak_source": "%d SMs x %d FP32 lanes x %.0f MHz (sm_max_mhz from %s)" % (
                    SM_COUNT, FP32_LANES_PER_SM, sm_max_mhz, peak_src),
                "traffic": traffic, "traffic_unit": "bytes per launch", "traffic_source": traffic_src,
                "frac_at_observed_clock": (achieved / fp32_peak) * sm_max_mhz / clocks["sm_mhz"]
                if clocks and clocks.get("sm_mhz") else None,
            },
            "e2e": {"value": aggregate_rate(1 if sharded else world, e2e_steps, e2e_s), "unit": "steps/s", "h2d_bytes_per_step": 72 * N,
                    "d2h_bytes_per_step": 72 * N, "steps": e2e_steps,
                    "what": "independent one-step requests through the C ABI, every step: pasta_set_state_host_async(x,v,F) "
                            "[pinned host -> device] + pasta_step(1) + pasta_get_state_host_async(x,v,F) [device -> pinned "
                            "host]; the library pipelines the copies on two side streams (double-buffered staging); "
                            "pasta_host_sync at the end, inside the timed region",
                    "serial_feedback_chain": {
                        "value": aggregate_rate(1 if sharded else world, e2e_steps, e2e_serial_s), "unit": "steps/s",
                        "what": "pasta_set_state_host + pasta_step(1) + pasta_get_state_host with the result fed back as the "
                                "next input (blocking; copies and compute strictly serial)"}},
            "gpu_launches": launches, "wall_s": t_wall, "clocks": clocks,
            "energies_MeV": {"KE": ke, "PE": pe},
        }
        if args.config == 4 and not args.no_config2 and world == 1:
            line["config2"] = config2_block(args, flush, barrier, local_rank, fp32_peak)
        if not args.no_cpu_baseline and world == 1:
            # the oracle gets the state the simulation ended in, so that its FP64 PE and the GPU's are of ONE configuration
            xs, vs, ps, Ls, _ = sim.get_state()
            ke_end, pe_end = sim.energy()
            state = (xs.cpu().numpy(), vs.cpu().numpy(), ps.cpu().numpy(), Ls)
            line["cpu_baseline"] = cpu_baseline(args.config, args.cpu_budget, state=state)
            pe_fp64 = line["cpu_baseline"]["PE_MeV"]
            rel = abs(pe_end - pe_fp64) / abs(pe_fp64)
            line["pe_parity"] = {"gpu_PE_MeV": pe_end, "oracle_fp64_PE_MeV": pe_fp64, "rel": rel, "gate": 1e-6, "ok": bool(rel <= 1e-6),
                                 "what": "total PE of all %d nucleons of the final state of this run: the CUDA path against "
                                         "orc_forces_cells" % N}
        print(json.dumps(line), flush=True)
    sim.close()
    if dist is not None:
        dist.destroy_process_group()


def run_sweep(args):
    """--sweep 3|5: the whole decompression run of BASELINE config 3 or 5 (20 000 steps, n = 0.08 -> 0.00125 fm^-3),
    timed in chunks of --sweep-chunk steps with CUDA events -- steps/s against density, the axis of the paper's
    Fig. 1/2 -- then friends-of-friends clustering at r_cl = 3 fm and the composition summary.
    One JSON line."""
    import torch

    import paper_1412_8502_b200 as pasta

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    c = inputs.CONFIGS[args.sweep]
    prm = pasta.default_params(r_c=c["r_c"], thermostat_interval=c["thermostat_interval"],
                               scale_per_step=c["scale_per_step"])
    sim = pasta.Sim(c["N"], c["Y_P"], c["density"], c["T"], params=prm, seed=1)
    pts, done = [], 0
    sm_max_mhz, _, _ = peaks()
    fp32_peak = SM_COUNT * FP32_LANES_PER_SM * sm_max_mhz * 1e6
    n_brk = 10  # steps at the end of every chunk that run with the library's event brackets on (K2 time for the roofline)
    t_all0 = time.perf_counter()
    while done < c["steps"]:
        n = min(args.sweep_chunk, c["steps"] - done)
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        sim.step(n - n_brk, c["dt"])
        b.record()
        sim.set_timing(True)
        sim.step(n_brk, c["dt"])
        tm = sim.get_timing()
        sim.set_timing(False)
        torch.cuda.synchronize()
        done += n
        L = sim.box_length()
        ke, pe = sim.energy()
        pairs, pairs_nz = sim.pair_counts()
        k2_s = tm["force_ms"] * 1e-3 / max(1, tm["force_evals"])
        work = 17.0 * pairs_nz + 8.0 * c["Y_P"] ** 2 * pairs  # as in the headline: only pairs with a non-zero FP32 term
        pts.append({"step": done, "L_fm": L, "density": c["N"] / L ** 3, "steps_per_s": 1e3 * (n - n_brk) / a.elapsed_time(b),
                    "PE_per_nucleon": pe / c["N"], "T_kin": ke / (1.5 * c["N"]),
                    "ordered_pairs": pairs, "nonzero_pairs": pairs_nz, "k2_ms": 1e3 * k2_s,
                    "roofline": {"bound": "alu", "frac": work / k2_s / fp32_peak, "achieved": work / k2_s / 1e9,
                                 "peak": fp32_peak / 1e9, "unit": "G FP32 lane-instr/s, work performed"}})
    wall = time.perf_counter() - t_all0
    list_stats = sim.list_stats()
    t0 = time.perf_counter()
    label, ncl = sim.clusters(c["r_cl"])
    A, Z = sim.cluster_sizes()
    comp = sim.composition(12)
    torch.cuda.synchronize()
    fof_s = time.perf_counter() - t0
    # the paper's own two-radius MST clusters on the same final configuration
    _, ncl_mst = sim.clusters_mst(4.5, 3.0)
    comp_mst = sim.composition(12)
    A = A.cpu().numpy()
    Z = Z.cpu().numpy()
    heavy = A >= 12
    import numpy as np

    hist = {}
    for a_, z_ in zip(A[heavy].tolist(), Z[heavy].tolist()):
        hist[(a_ // 20 * 20, z_ // 10 * 10)] = hist.get((a_ // 20 * 20, z_ // 10 * 10), 0) + 1
    line = {"sweep": args.sweep, "workload": workload_config(args.sweep, 1)["workload"] + ", decompression to 0.00125 fm^-3",
            "steps": c["steps"], "wall_s": wall, "list_stats": list_stats, "points": pts, "clusters": ncl, "fof_s": fof_s, "composition": comp,
            "mst_r_pp_4.5_r_np_3.0": {"clusters": ncl_mst, "composition": comp_mst}, "largest_A": int(A.max()), "AZ_histogram_A20_Z10_bins": {"%d,%d" % k: v for k, v in sorted(hist.items())}}
    print(json.dumps(line), flush=True)
    sim.close()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=500)
    ap.add_argument("--warmup", type=int, default=20)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=4, choices=[2, 4])
    ap.add_argument("--sweep", type=int, default=0, choices=[0, 3, 5],
                    help="run the whole decompression of config 3 or 5 and report steps/s against density")
    ap.add_argument("--sweep-chunk", type=int, default=1000)
    ap.add_argument("--shard", action="store_true", help="with --gpus N > 1: one simulation sharded by targets over the N "
                    "GPUs (strong scaling) instead of N independent replicas")
    ap.add_argument("--seed", type=int, default=1, help="seed of the synthetic start (rank r uses seed + r)")
    ap.add_argument("--params", default="", help="comma-separated pasta_params overrides: a second reported mode, "
                    "e.g. r_nuc=11.5 (the paper's range split) or skip_exact_zeros=0")
    ap.add_argument("--cpu-budget", type=float, default=15.0, help="seconds of oracle time for cpu_baseline")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-config2", action="store_true", help="leave the 51 200-nucleon block out of the config-4 line")
    args = ap.parse_args()
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if args.sweep:
        if rank == 0:
            run_sweep(args)
    elif args.impl == "reference":
        run_reference(args, rank, world)
    else:
        run_ours(args, rank, world, local_rank)


if __name__ == "__main__":
    main()
