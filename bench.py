#!/usr/bin/env python
"""bench.py -- one JSON line for the CLOSURE hot path on B200 (contract: see DESIGN.md "Measurement").

    python bench.py --gpus N --steps K --warmup W            # this build (CUDA path via the C ABI)
    python bench.py --impl reference --steps K --warmup W    # the CPU oracle on the host cores

A "step" is one pass of the whole hot path over one synthetic instance batch: walker kernel
(a0-a7) + compaction kernel (a8), device-resident, timed with CUDA events; the host MEGB (a9)
is timed separately and is inside the end-to-end number.  The workload at one
GPU is BASELINE.json configs[1] (C2: 3D registration, N=50, 65,536 walkers x 1,000 iterations).
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np

from paper_2403_09990_b200 import instances as I

METRIC = "walker_steps_per_sec"
UNIT = "walker-steps/s"
WALK_SEED = 42

# Arithmetic of the walker kernel's inner loops (FMA = 2), multiplied by the executed
# counts the kernel reports (closure_get_stats):
#   one (pose, constraint) pair  = 3 FMA + 1 compare/max                      = 7   (fp32, or fp64 where it falls back)
#   one per-constraint set-up    = R a (6 FMA + 3 MUL) + 6 ADD/SUB + |u|^2 (2 FMA + MUL) = 26 (+1 on the ladder), fp64
FLOP_PAIR, FLOP_SETUP_A, FLOP_SETUP_L = 7.0, 26.0, 27.0
# reprojection residual: eq. (14) pair = 4 FMA + RCP + 3 MUL + max = 13; cone pair = 8 FMA + max = 17
FLOP_PAIR_REPROJ_A, FLOP_PAIR_REPROJ_L = 13.0, 17.0
# DRAM traffic of the walker kernel per launch (dram__bytes_read.sum + dram__bytes_write.sum) from the committed
# `ncu --set full` captures of this very command line: profiles/r1_v6_final_ncu.md (C2, default arguments)
# and profiles/r1_v4_reproj_megb_ncu.md (--config 3).  Other workloads have no capture: null.
NCU_TRAFFIC_BYTES = {("C2_reg_n50", "rot", 64): 500480 + 63744, ("C3_reproj_n8", "rot", 64): 549376 + 776448}


def _params_dict(P) -> dict:
    return dict(mode="ROT" if P.mode == 0 else "TRANS", N_P=P.n_p, N_P_star=P.n_p_star, N_T=P.n_t,
                gamma=P.gamma, omega0=P.omega0, v0=P.v0, t_p=P.t_p, theta_p=P.theta_p)


def _workload(config: int):
    inst = I.make_instance(config)
    S0 = I.make_init_poses(inst, 128)
    return inst, S0


# ------------------------------------------------------------------------------- clocks
class ClockSampler:
    """nvidia-smi clocks and throttle reasons DURING the timed region (B200_PROFILING.md)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                 "-lms", "200"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            threading.Thread(target=self._pump, daemon=True).start()
        except OSError:
            self.proc = None

    def _pump(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        sm, mx, reasons = [], [], set()
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1]))
            except (ValueError, IndexError):
                continue
            for name, val in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[3:7]):
                if val.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


# ------------------------------------------------------------------------------- oracle legs
def _oracle_leg(inst, S0, walkers: int, steps: int, threads: int, seed: int) -> float:
    import oracle
    ids = np.arange(walkers, dtype=np.int64) * max(1, inst.num_walkers // walkers)   # strided subset
    t0 = time.perf_counter()
    oracle.walk(inst, inst.params, S0, ids, steps, seed, n_threads=threads)
    return time.perf_counter() - t0


def _sample_size(inst, S0, threads: int, target_s: float) -> int:
    """Walkers for about target_s seconds of oracle time, from a short calibration leg."""
    steps = max(1, min(inst.num_steps, 50))
    dt = _oracle_leg(inst, S0, threads, steps, threads, WALK_SEED + 7)
    rate = threads * steps / max(dt, 1e-6)                      # walker-steps/s
    return int(min(inst.num_walkers, max(threads, round(target_s * rate / inst.num_steps))))


def cpu_baseline(inst, S0) -> dict:
    """The oracle as it stands on the host cores, on a bounded sample of the same workload."""
    import oracle
    oracle.build()
    threads = os.cpu_count() or 1
    walkers = _sample_size(inst, S0, threads, 15.0)
    dt = _oracle_leg(inst, S0, walkers, inst.num_steps, threads, WALK_SEED)
    return {"value": walkers * inst.num_steps / dt, "unit": UNIT, "cores": threads, "kind": "oracle",
            "sample": f"{walkers} strided walkers x {inst.num_steps} iterations of the same instance, "
                      f"OpenMP over walkers, {dt:.2f} s wall"}


def run_reference(args) -> None:
    """--impl reference: the oracle timed on the host cores (rank 0 only)."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    import oracle
    oracle.build()
    inst, S0 = _workload(args.config)
    if args.mode == "trans":
        inst.params.mode = I.MODE_TRANS
    threads = os.cpu_count() or 1
    P = inst.params
    walkers = _sample_size(inst, S0, threads, 60.0 / max(1, args.steps))
    for w in range(args.warmup):
        _oracle_leg(inst, S0, max(threads, walkers // 8), max(1, inst.num_steps // 8), threads, WALK_SEED + w)
    t0 = time.perf_counter()
    for k in range(args.steps):
        _oracle_leg(inst, S0, walkers, inst.num_steps, threads, WALK_SEED + k)
    dt = time.perf_counter() - t0
    value = args.steps * walkers * inst.num_steps / dt
    sample = f"per step: {walkers} strided walkers x {inst.num_steps} iterations (of {inst.num_walkers} walkers)"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": inst.name, "N": inst.n, "walkers": inst.num_walkers, "iterations": inst.num_steps,
                   "params": _params_dict(P), "S0": 128},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


# ------------------------------------------------------------------------------- this build
def run_cuda(args) -> None:
    import torch
    import torch.distributed as dist
    from paper_2403_09990_b200 import binding as B

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the CUDA path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    if not os.path.exists(B.LIB_PATH):      # a checkout without the built library (git-ignored): compile it once
        if rank == 0:
            from paper_2403_09990_b200 import build as build_mod
            build_mod.build_library()
        if world > 1:
            dist.barrier()
    B.load_library()     # fails loudly if libclosure_b200.so is missing

    inst, S0 = _workload(args.config)
    P = inst.params
    W, S, nb = inst.num_walkers, inst.num_steps, inst.batch
    insts = [inst] if nb == 1 else [I.make_instance(args.config, b) for b in range(nb)]
    S0s = [S0] if nb == 1 else [I.make_init_poses(it, 128) for it in insts]
    # Weak scaling: every rank walks W walkers per instance with its own
    # walker-id range [rank*W, (rank+1)*W); walkers are independent, no collective
    # sits on the data path.
    begin = rank * W
    handles = []
    if args.precision == 32:
        for it in insts:
            it.params.precision = 32
    if args.mode == "trans":
        if not (P.v0 > 0.0 and P.theta_p > 0.0):
            raise SystemExit("--mode trans needs v0 > 0 and theta_p > 0 (BASELINE config 3)")
        for it in insts:
            it.params.mode = I.MODE_TRANS
    for it, s0 in zip(insts, S0s):
        h = B.Closure.closure_create(it)
        h.closure_set_init(s0)
        handles.append(h)
    dev = torch.device("cuda", local)
    samples = torch.empty((nb * W, 12), dtype=torch.float64, device=dev)
    flags = torch.empty((nb * W,), dtype=torch.uint8, device=dev)
    compacted = torch.empty((nb * W, 12), dtype=torch.float64, device=dev)
    count = torch.zeros((1,), dtype=torch.int64, device=dev)
    flush = torch.empty((256 << 20,), dtype=torch.uint8, device=dev)      # > 126 MB L2
    stream = torch.cuda.current_stream()

    def walk(seed):
        if nb == 1:
            handles[0].closure_sample(W, S, seed, samples, flags, stream, walker_begin=begin)
        else:
            B.closure_sample_batch(handles, W, S, [seed + 1000 * b for b in range(nb)],
                                   samples.view(nb, W, 12), flags.view(nb, W), stream)

    def step(seed, ev=None):
        if ev:
            ev[0].record(stream)
        walk(seed)
        if ev:
            ev[1].record(stream)
        handles[0].closure_compact(samples, flags, compacted, count, stream)
        if ev:
            ev[2].record(stream)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    peak64, _ = B.closure_alu_peak(64)
    peak32, _ = B.closure_alu_peak(32)
    peak_philox, _ = B.closure_alu_peak(4)          # Philox4x32-10 calls per second
    for w in range(args.warmup):
        step(WALK_SEED + 100 + w)
        flush.fill_(w)
    barrier()
    clocks = ClockSampler(local)
    clocks.start()
    evs = [[torch.cuda.Event(enable_timing=True) for _ in range(3)] for _ in range(args.steps)]
    t_begin, t_end = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    t_begin.record(stream)
    for k in range(args.steps):
        step(WALK_SEED + k, evs[k])
        flush.fill_(k)                                                     # L2 flush between iterations
    t_end.record(stream)
    barrier()
    clk = clocks.stop()
    total_ms = t_begin.elapsed_time(t_end)
    if world > 1:
        tt = torch.tensor([total_ms], dtype=torch.float64, device=dev)
        dist.all_reduce(tt, op=dist.ReduceOp.MAX)
        total_ms = float(tt.item())
    walk_ms = [e[0].elapsed_time(e[1]) for e in evs]
    comp_ms = [e[1].elapsed_time(e[2]) for e in evs]
    units = float(world) * nb * W * S * args.steps
    value = units / (total_ms * 1e-3)

    out = None
    if rank == 0:
        # executed work of one step (deterministic: same seed as timed step 0), counted by an untimed launch
        handles[0].closure_enable_stats(True)
        walk(WALK_SEED)
        st = handles[0].closure_get_stats()
        handles[0].closure_enable_stats(False)
        # the kernel decides in fp32 with certified error bounds and falls back to fp64:
        # executed arithmetic per pipe, and the time the two CUDA-core pipes need for it at their measured peaks
        fpa, fpl = (FLOP_PAIR_REPROJ_A, FLOP_PAIR_REPROJ_L) if inst.residual_type == 1 else (FLOP_PAIR, FLOP_PAIR)
        fsa, fsl = FLOP_SETUP_A, FLOP_SETUP_L
        if args.mode == "trans":
            # Alg. A8: every perturbation has its own rotation, a pair is one direct residual evaluation
            # (REG 26, REPROJ 31 + reciprocal, POSE_REG 36 flop); no shared set-up
            fpa = fpl = {1: 31.0, 2: 26.0}.get(inst.residual_type, 36.0)
            fsa = fsl = 0.0
        flops64 = fpa * st["perturb_pairs"] + fpl * st["ladder_pairs"] + fsa * st["perturb_setups"] \
            + fsl * st["ladder_setups"]
        flops32 = fpa * st["perturb_pairs_f32"] + fpl * st["ladder_pairs_f32"]
        flops = flops64 + flops32
        walk_s = statistics.mean(walk_ms) * 1e-3
        achieved = flops / walk_s / 1e12
        t_min = flops64 / peak64 + flops32 / peak32
        peak_mix = flops / t_min / 1e12
        nom_mhz = float(clk.get("sm_max_mhz") or 1965.0)
        nom32, nom64 = 148 * 128 * 2 * nom_mhz * 1e6, 148 * 64 * 2 * nom_mhz * 1e6
        # the integer work a flop count does not see: one Philox4x32-10 call per perturbation and iteration
        philox_calls = float(st["walker_steps"]) * (P.n_p + 1)
        t_min_rng = t_min + philox_calls / peak_philox
        nominal_pairs = (P.n_p + P.n_p_star * P.n_t) * inst.n
        n_cnt = int(count.item())
        comp_bytes = nb * W * 1 + n_cnt * 96 * 2
        comp_s = statistics.mean(comp_ms) * 1e-3
        peaks = {}
        try:
            peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
        except OSError:
            pass
        hbm_peak = float(peaks.get("hbm_gbs", 6650.0))

        # end to end through the C ABI with HOST buffers: create + set_init (H2D) + walk + compact +
        # D2H of the compacted cloud + host MEGB, every step.
        e2e_steps = max(1, min(args.steps, 3))
        megb_s, d2h = [], 0
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        for k in range(e2e_steps):
            hs = []
            for it, s0 in zip(insts, S0s):
                h = B.Closure.closure_create(it)
                h.closure_set_init(s0)
                hs.append(h)
            for b, h in enumerate(hs):
                r = h.closure_run(W, S, WALK_SEED + k + 1000 * b, stream)
                megb_s.append(r["host_seconds"])
                d2h += r["count"] * 96 + 8
                h.closure_destroy()
        torch.cuda.synchronize()
        e2e_dt = time.perf_counter() - t0
        h2d = sum(it.measurements.nbytes + it.betas.nbytes + s0.nbytes + 256 for it, s0 in zip(insts, S0s))

        # Step I on the device (not part of the timed step): trials -> compaction -> S_0 for
        # 1,000 trials end to end, and the trial kernel alone at the 100,000 trials of the paper's pure-RANSAG
        # comparison.  Ex.1: P3P trials; Ex.2: Arun; Ex.3: convex combinations.
        hs1 = B.Closure.closure_create(insts[0])
        t_s1 = []
        for k in range(12):
            t1 = time.perf_counter()
            n0_s1 = hs1.closure_init_from_trials(1000, WALK_SEED + k, 128, stream)
            t_s1.append(1e3 * (time.perf_counter() - t1))
        p_s1 = torch.empty((100000, 12), dtype=torch.float64, device=dev)
        o_s1 = torch.empty((100000,), dtype=torch.uint8, device=dev)
        k_s1 = []
        for k in range(6):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            hs1.closure_init_sample(100000, WALK_SEED + k, p_s1, o_s1, stream)
            e1.record(stream)
            torch.cuda.synchronize()
            k_s1.append(e0.elapsed_time(e1))
        step1 = {"ms_1000_trials_to_S0_end_to_end": statistics.median(t_s1[2:]), "S0_size": n0_s1,
                 "kernel_ms_100000_trials": statistics.median(k_s1[1:]),
                 "accepted_fraction": float(o_s1.float().mean().item())}
        hs1.closure_destroy()
        del p_s1, o_s1

        fp32_report = None
        if args.precision == 32:
            # measured difference of the fp32 mode from the fp64 path: same instance, same seed, decision traces
            import copy
            Wc = min(W, 16384)
            P64 = copy.copy(insts[0].params)
            P64.precision = 64
            h64 = B.Closure.closure_create(insts[0], P64)
            h64.closure_set_init(S0s[0])
            s32, f32_, t32 = handles[0].closure_sample(Wc, S, WALK_SEED, trace=True)
            s64, f64_, t64 = h64.closure_sample(Wc, S, WALK_SEED, trace=True)
            same = (t32 == t64).all(dim=1)
            c32, n32 = handles[0].closure_compact(s32, f32_)
            r32 = handles[0].closure_megb(c32, int(n32.item()))
            c64, n64 = h64.closure_compact(s64, f64_)
            r64 = h64.closure_megb(c64, int(n64.item()))
            fp32_report = {"walkers_compared": Wc, "iterations": S,
                           "walkers_with_identical_decisions": float(same.float().mean().item()),
                           "max_abs_sample_difference_among_those": float((s32[same] - s64[same]).abs().max().item())
                           if bool(same.any()) else None,
                           "rot_radius_rel_diff": abs(r32["rot_radius"] - r64["rot_radius"]) / r64["rot_radius"],
                           "trans_radius_rel_diff": abs(r32["trans_radius"] - r64["trans_radius"]) / r64["trans_radius"]}
            h64.closure_destroy()
            del s32, s64, t32, t64

        # the compaction kernel alone at BASELINE config 5's size (4,194,304 walkers, every sample kept):
        # the size at which it is HBM-bound rather than launch-bound
        nbig = 4194304
        big_s = torch.empty((nbig, 12), dtype=torch.float64, device=dev).fill_(1.0)
        big_f = torch.ones((nbig,), dtype=torch.uint8, device=dev)
        big_o = torch.empty_like(big_s)
        big_ms = []
        for k in range(7):
            flush.fill_(k)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            handles[0].closure_compact(big_s, big_f, big_o, count, stream)
            e1.record(stream)
            torch.cuda.synchronize()
            if k >= 2:
                big_ms.append(e0.elapsed_time(e1))
        big_bytes = nbig * 1 + int(count.item()) * 96 * 2
        big_gbs = big_bytes / (statistics.mean(big_ms) * 1e-3) / 1e9
        del big_s, big_f, big_o

        # per-instance latency at the paper's own scale (|S_0| N_W = 200 walks, N_I = 5):
        # host buffers in, MEGB out, through closure_create + closure_set_init + closure_run
        small_ms = []
        for k in range(25):
            t1 = time.perf_counter()
            h = B.Closure.closure_create(insts[0])
            h.closure_set_init(S0s[0])
            h.closure_run(200, 5, WALK_SEED + k, stream)
            h.closure_destroy()
            small_ms.append(1e3 * (time.perf_counter() - t1))
        small_ms = statistics.median(small_ms[5:])

        out = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": total_ms / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None,
            "dtype": "f64" if args.precision == 64 else "f32 decisions, f64 poses", "data": "synthetic",
            "config": {"workload": inst.name, "residual": "3D registration" if inst.residual_type == 2 else
                       ("2D reprojection" if inst.residual_type == 1 else "pose regression"),
                       "N": inst.n, "walkers": W, "iterations": S, "instances": nb, "S0": 128,
                       "params": _params_dict(P), "l2": "256 MiB buffer written between timed iterations",
                       "sharding": "walker ranges per rank, no collective"},
            "constraint_evals_per_sec_nominal": value * nominal_pairs,
            "constraint_evals_per_sec_executed": (st["perturb_pairs"] + st["ladder_pairs"] + st["perturb_pairs_f32"]
                                                  + st["ladder_pairs_f32"]) / walk_s * world,
            "latency_ms": {"walker_kernel": statistics.mean(walk_ms), "compaction_kernel": statistics.mean(comp_ms),
                           "megb": 1e3 * statistics.median(megb_s), "megb_max": 1e3 * max(megb_s), "e2e_per_instance": 1e3 * e2e_dt / (e2e_steps * nb),
                           "e2e_200_walkers_x_5_iterations": small_ms},
            "boundary_fraction": n_cnt / float(nb * W),
            "roofline": {"bound": "alu", "kernel": "walker_coop_trans_kernel" if args.mode == "trans" else
                         ("walker_coop_reproj_kernel" if inst.residual_type == 1 else "walker_coop_kernel"),
                         "achieved": achieved, "peak": peak_mix, "unit": "TFLOP/s", "frac": achieved / peak_mix,
                         "traffic": NCU_TRAFFIC_BYTES.get((inst.name, args.mode, args.precision)),
                         "peak_source": "executed flops / (fp64 flops / DFMA peak + fp32 flops / FFMA peak), both peaks "
                                        "measured in this run by closure_alu_peak (register-resident FMA chains)",
                         "fp32": {"flops_per_launch": flops32, "achieved": flops32 / walk_s / 1e12, "peak": peak32 / 1e12},
                         "fp64": {"flops_per_launch": flops64, "achieved": flops64 / walk_s / 1e12, "peak": peak64 / 1e12},
                         "flops_per_launch": flops,
                         # the unit-count peak of SURVEY.md 8(d): 148 SMs x 128 FP32 (64 FP64) lanes x 2 x the maximum SM clock
                         "frac_of_nominal": (flops32 / nom32 + flops64 / nom64) / walk_s,
                         "peak_nominal": {"fp32": nom32 / 1e12, "fp64": nom64 / 1e12, "sm_mhz": nom_mhz},
                         "philox": {"calls_per_launch": philox_calls, "peak_calls_per_s": peak_philox,
                                    "note": "Philox4x32-10 calls at the rate of a kernel that does nothing else"},
                         "frac_incl_philox": t_min_rng / walk_s,
                         "executed_pairs_per_walker_step": (st["perturb_pairs"] + st["ladder_pairs"] + st["perturb_pairs_f32"]
                                                            + st["ladder_pairs_f32"]) / st["walker_steps"],
                         "fp64_fallback_steps": st["fallback_steps"] / st["walker_steps"],
                         "accepted_steps": st["accepted_steps"] / st["walker_steps"]},
            "roofline_compaction": {"bound": "hbm", "kernel": "compact_kernel", "achieved": comp_bytes / comp_s / 1e9,
                                    "peak": hbm_peak, "unit": "GB/s", "frac": comp_bytes / comp_s / 1e9 / hbm_peak,
                                    "bytes_per_launch": comp_bytes, "peak_source": "MEASURED_PEAKS.json hbm_gbs"
                                    if peaks else "fallback 6650",
                                    "at_4194304_walkers": {"achieved": big_gbs, "frac": big_gbs / hbm_peak,
                                                           "bytes_per_launch": big_bytes,
                                                           "ms": statistics.mean(big_ms)}},
            "e2e": {"value": e2e_steps * nb * W * S / e2e_dt, "unit": UNIT, "h2d_bytes_per_step": h2d,
                    "d2h_bytes_per_step": d2h // e2e_steps},
            "gpu_launches": args.steps * (-(-nb // 96) + 1),     # walker launch(es) + compaction kernel per step
            "clocks": clk,
        }
        if fp32_report is not None:
            out["fp32_mode"] = fp32_report
        if step1 is not None:
            out["step1"] = step1
        if not args.no_cpu_baseline and world == 1:
            out["cpu_baseline"] = cpu_baseline(inst, S0)
    for h in handles:
        h.closure_destroy()
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()
    if out is not None:
        print(json.dumps(out))


def main() -> None:
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="cuda", choices=["cuda", "reference"])
    ap.add_argument("--config", type=int, default=2, help="BASELINE.json config 1..5 (default 2 = configs[1])")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--mode", default="rot", choices=["rot", "trans"],
                    help="rot: Alg. 2, the rotation-boundary sampler (default); trans: Alg. A8, the translation-boundary "
                         "sampler (config 3 carries the paper's v0 and theta_p; other configs have v0 = 0)")
    ap.add_argument("--precision", type=int, default=64, choices=[64, 32],
                    help="64: every decision is the fp64 decision (default, the parity path); 32: fp32 mode, with its "
                         "measured difference from the fp64 path in the output")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_cuda(args)


if __name__ == "__main__":
    main()
