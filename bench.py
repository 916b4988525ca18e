#!/usr/bin/env python
"""bench.py -- one JSON line for the CLOSURE hot path on B200 (contract: see DESIGN.md "Measurement").

    python bench.py --gpus N --steps K --warmup W            # this build (CUDA path via the C ABI)
    python bench.py --impl reference --steps K --warmup W    # the CPU oracle on the host cores

A "step" is one pass of the whole hot path over one synthetic instance batch: walker kernel
(a0-a7) + compaction kernel (a8), device-resident, timed with CUDA events; the MEGB (a9) is timed
separately and is inside the end-to-end number.  The workload at one GPU is the largest
single-GPU configuration of BASELINE.json, configs[4] (C5: 3D registration, N=200, a batch of 64
instances x 65,536 walkers x 2,000 iterations); the same line carries one short measurement of every
other config (`per_config`), the regime the paper itself runs (`moving_regime`: N_I = 5 and 20,
PAPER.md:374, 440, 508) and the per-component latency split of Table IV.
"""
from __future__ import annotations

import argparse
import hashlib
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
DTYPE = "f64 results (certified f32 screening, f64 fall-back)"

# Arithmetic of the walker kernel's inner loops (FMA = 2), multiplied by the executed
# counts the kernel reports (closure_get_stats):
#   one (pose, constraint) pair  = 3 FMA + 1 compare/max                      = 7   (fp32, or fp64 where it falls back)
#   one per-constraint set-up    = R a (6 FMA + 3 MUL) + 6 ADD/SUB + |u|^2 (2 FMA + MUL) = 26 (+1 on the ladder), fp64
FLOP_PAIR, FLOP_SETUP_A, FLOP_SETUP_L = 7.0, 26.0, 27.0
# reprojection residual: eq. (14) pair = 4 FMA + RCP + 3 MUL + max = 13; cone pair = 8 FMA + max = 17
FLOP_PAIR_REPROJ_A, FLOP_PAIR_REPROJ_L = 13.0, 17.0
# DRAM traffic of the walker kernel per launch (dram__bytes_read.sum + dram__bytes_write.sum) from the committed
# `ncu --set full` captures under profiles/ (profiles/ncu_traffic.json), valid only for the kernel sources they
# were taken on: each entry carries the hash of csrc/ at capture time (_csrc_hash) and reads as null once the
# sources differ.
NCU_TRAFFIC_BYTES: dict = {}
try:
    with open(os.path.join(ROOT, "profiles", "ncu_traffic.json")) as _f:
        NCU_TRAFFIC_BYTES = json.load(_f)
except (OSError, ValueError):
    pass

# the other configs measured in the same line: (config, mode)
PER_CONFIG = [(1, "rot"), (2, "rot"), (3, "rot"), (3, "trans"), (4, "rot")]
RESIDUAL_NAME = {1: "2D reprojection", 2: "3D registration", 3: "pose regression", 4: "pose regression (split)"}


def _csrc_hash() -> str:
    h = hashlib.sha256()
    d = os.path.join(ROOT, "paper_2403_09990_b200", "csrc")
    for name in sorted(os.listdir(d)):
        if name.endswith((".cu", ".cuh", ".h", ".cpp")):
            with open(os.path.join(d, name), "rb") as f:
                h.update(name.encode() + b"\0" + f.read())
    return h.hexdigest()[:16]


def _traffic(workload: str, mode: str, precision: int, walkers: int, iterations: int, instances: int):
    """DRAM bytes of the walker launch from the committed capture of this very launch (same sources, same size), else None."""
    e = NCU_TRAFFIC_BYTES.get(f"{workload}/{mode}/{precision}")
    if not e or e.get("csrc_hash") != _csrc_hash():
        return None
    if (e.get("walkers"), e.get("iterations"), e.get("instances")) != (walkers, iterations, instances):
        return None
    return e.get("bytes")


def _params_dict(P) -> dict:
    return dict(mode="ROT" if P.mode == 0 else "TRANS", N_P=P.n_p, N_P_star=P.n_p_star, N_T=P.n_t,
                gamma=P.gamma, omega0=P.omega0, v0=P.v0, t_p=P.t_p, theta_p=P.theta_p)


def _config_dict(inst, W, S, nb, sharding: str) -> dict:
    return {"workload": inst.name, "residual": RESIDUAL_NAME.get(inst.residual_type, str(inst.residual_type)),
            "N": inst.n, "walkers": W, "iterations": S, "instances": nb, "S0": 128,
            "params": _params_dict(inst.params), "l2": "256 MiB buffer written between timed iterations",
            "sharding": sharding}


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
        sm, mx, pw, reasons = [], [], [], set()
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1])); pw.append(float(r[2]))
            except (ValueError, IndexError):
                continue
            for name, val in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[3:7]):
                if val.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


# ------------------------------------------------------------------------------- oracle legs
def _oracle_leg(inst, S0, walkers: int, steps: int, threads: int, seed: int):
    import oracle
    ids = np.arange(walkers, dtype=np.int64) * max(1, inst.num_walkers // walkers)   # strided subset
    t0 = time.perf_counter()
    out = oracle.walk(inst, inst.params, S0, ids, steps, seed, n_threads=threads)
    return time.perf_counter() - t0, out


def _sample_size(inst, S0, threads: int, target_s: float) -> int:
    """Walkers for about target_s seconds of oracle time, from a short calibration leg."""
    steps = max(1, min(inst.num_steps, 200))
    cal = 4 * threads                                           # enough walkers per thread to amortise the thread start-up
    dt, _ = _oracle_leg(inst, S0, cal, steps, threads, WALK_SEED + 7)
    rate = cal * steps / max(dt, 1e-6)                          # walker-steps/s
    return int(min(inst.num_walkers, max(threads, round(target_s * rate / inst.num_steps))))


def cpu_baseline(inst, S0) -> dict:
    """The oracle as it stands on the host cores, on a bounded sample of the same workload:
    OpenMP over walkers on all cores, one thread alone, and the oracle's own miniball on the samples it produced."""
    import oracle
    oracle.build()
    P = inst.params
    nominal = (P.n_p + P.n_p_star * P.n_t) * inst.n           # Alg. 3's dense count per walker-step
    threads = os.cpu_count() or 1
    walkers = _sample_size(inst, S0, threads, 12.0)
    dt, (smp, flg) = _oracle_leg(inst, S0, walkers, inst.num_steps, threads, WALK_SEED)
    w1 = max(1, _sample_size(inst, S0, 1, 5.0))
    dt1, _ = _oracle_leg(inst, S0, w1, inst.num_steps, 1, WALK_SEED)
    t0 = time.perf_counter()
    cloud = oracle.compact(smp, flg)
    if len(cloud):
        oracle.megb(cloud, oracle.mean_pose(S0)[0])
    dtm = time.perf_counter() - t0
    value = walkers * inst.num_steps / dt
    return {"value": value, "unit": UNIT, "cores": threads, "kind": "oracle",
            "sample": f"{walkers} strided walkers x {inst.num_steps} iterations of instance 0 of the same workload, "
                      f"OpenMP over walkers, {dt:.2f} s wall",
            "constraint_evals_per_sec_nominal": value * nominal,
            "single_thread": {"value": w1 * inst.num_steps / dt1, "unit": UNIT, "cores": 1,
                              "constraint_evals_per_sec_nominal": w1 * inst.num_steps / dt1 * nominal,
                              "sample": f"{w1} strided walkers x {inst.num_steps} iterations, {dt1:.2f} s wall"},
            "host_miniball_ms": 1e3 * dtm,
            "host_miniball_sample": f"oracle compaction + MEGB (Welzl) of the {len(cloud)} boundary samples of the OpenMP leg",
            "nproc": os.cpu_count()}


def run_reference(args) -> None:
    """--impl reference: the oracle timed on the host cores (rank 0 only)."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    import oracle
    oracle.build()
    inst, S0 = _workload(args.config)
    if args.mode == "trans":
        inst.params.mode = I.MODE_TRANS
    if args.iterations:
        inst.num_steps = args.iterations
    if args.walkers:
        inst.num_walkers = args.walkers
    threads = os.cpu_count() or 1
    walkers = _sample_size(inst, S0, threads, 60.0 / max(1, args.steps))
    for w in range(args.warmup):
        _oracle_leg(inst, S0, max(threads, walkers // 8), max(1, inst.num_steps // 8), threads, WALK_SEED + w)
    t0 = time.perf_counter()
    for k in range(args.steps):
        _oracle_leg(inst, S0, walkers, inst.num_steps, threads, WALK_SEED + k)
    dt = time.perf_counter() - t0
    value = args.steps * walkers * inst.num_steps / dt
    sample = (f"per step: {walkers} strided walkers x {inst.num_steps} iterations of instance 0 "
              f"(of {inst.batch} instances x {inst.num_walkers} walkers)")
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": _config_dict(inst, inst.num_walkers, inst.num_steps, inst.batch, "walker ranges per rank, no collective"),
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


# ------------------------------------------------------------------------------- this build
class Workload:
    """Device-resident state of one (config, mode, precision) measurement: handles, output buffers, the launch."""

    def __init__(self, B, torch, config: int, mode: str, precision: int, begin: int = 0, walkers=None, iterations=None):
        self.B, self.torch = B, torch
        self.inst, self.S0 = _workload(config)
        self.config, self.mode, self.precision = config, mode, precision
        P = self.inst.params
        self.W = int(walkers or self.inst.num_walkers)
        self.S = int(iterations or self.inst.num_steps)
        self.nb = self.inst.batch
        self.insts = [self.inst] if self.nb == 1 else [I.make_instance(config, b) for b in range(self.nb)]
        self.S0s = [self.S0] if self.nb == 1 else [I.make_init_poses(it, 128) for it in self.insts]
        self.begin = begin
        if precision == 32:
            for it in self.insts:
                it.params.precision = 32
        if mode == "trans":
            if not (P.v0 > 0.0 and P.theta_p > 0.0):
                raise SystemExit("--mode trans needs v0 > 0 and theta_p > 0 (BASELINE config 3)")
            for it in self.insts:
                it.params.mode = I.MODE_TRANS
        self.handles = []
        for it, s0 in zip(self.insts, self.S0s):
            h = B.Closure.closure_create(it)
            h.closure_set_init(s0)
            self.handles.append(h)
        dev = torch.device("cuda", torch.cuda.current_device())
        n = self.nb * self.W
        self.samples = torch.empty((n, 12), dtype=torch.float64, device=dev)
        self.flags = torch.empty((n,), dtype=torch.uint8, device=dev)
        self.compacted = torch.empty((n, 12), dtype=torch.float64, device=dev)
        self.count = torch.zeros((1,), dtype=torch.int64, device=dev)
        self.stream = torch.cuda.current_stream()

    @property
    def kernel(self) -> str:
        if self.mode == "trans":
            return "walker_coop_trans_kernel"
        if self.inst.residual_type == 1:
            return "walker_coop_reproj_kernel"
        # N_P > 32: every perturbation against every constraint; N_P <= 32: best-first branch and bound
        return "walker_dense_kernel" if self.inst.params.n_p > 32 else "walker_coop_kernel"

    def walk(self, seed):
        B = self.B
        if self.nb == 1:
            self.handles[0].closure_sample(self.W, self.S, seed, self.samples, self.flags, self.stream,
                                           walker_begin=self.begin)
        else:
            B.closure_sample_batch(self.handles, self.W, self.S, [seed + 1000 * b for b in range(self.nb)],
                                   self.samples.view(self.nb, self.W, 12), self.flags.view(self.nb, self.W), self.stream)

    def step(self, seed, ev=None):
        if ev:
            ev[0].record(self.stream)
        self.walk(seed)
        if ev:
            ev[1].record(self.stream)
        self.handles[0].closure_compact(self.samples, self.flags, self.compacted, self.count, self.stream)
        if ev:
            ev[2].record(self.stream)

    def destroy(self):
        for h in self.handles:
            h.closure_destroy()
        self.handles = []
        self.samples = self.flags = self.compacted = None


def timed_steps(wl: Workload, steps: int, warmup: int, flush, barrier, seed0: int = WALK_SEED):
    """warmup untimed steps, then `steps` timed ones (CUDA events on the launching stream, an L2 flush between
    iterations) -> (total ms, [walker kernel ms], [compaction kernel ms])."""
    torch = wl.torch
    for w in range(warmup):
        wl.step(seed0 + 100 + w)
        flush.fill_(w)
    barrier()
    evs = [[torch.cuda.Event(enable_timing=True) for _ in range(3)] for _ in range(steps)]
    t_begin, t_end = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    t_begin.record(wl.stream)
    for k in range(steps):
        wl.step(seed0 + k, evs[k])
        flush.fill_(k)                                                     # L2 flush between iterations
    t_end.record(wl.stream)
    barrier()
    return (t_begin.elapsed_time(t_end), [e[0].elapsed_time(e[1]) for e in evs],
            [e[1].elapsed_time(e[2]) for e in evs])


def roofline_of(wl: Workload, walk_s: float, peaks: dict, seed: int = WALK_SEED) -> tuple[dict, dict]:
    """Executed work of one step (deterministic: the timed step's seed), counted by an untimed launch, against
    the CUDA-core peaks measured in this run."""
    inst, P = wl.inst, wl.inst.params
    h = wl.handles[0]
    h.closure_enable_stats(True)
    wl.walk(seed)
    st = h.closure_get_stats()
    h.closure_enable_stats(False)
    peak64, peak32, peak_philox, nom_mhz = peaks["f64"], peaks["f32"], peaks["philox"], peaks["nom_mhz"]
    # the kernel decides in fp32 with certified error bounds and falls back to fp64:
    # executed arithmetic per pipe, and the time the two CUDA-core pipes need for it at their measured peaks
    fpa, fpl = (FLOP_PAIR_REPROJ_A, FLOP_PAIR_REPROJ_L) if inst.residual_type == 1 else (FLOP_PAIR, FLOP_PAIR)
    fsa, fsl = FLOP_SETUP_A, FLOP_SETUP_L
    if wl.mode == "trans":
        # Alg. A8: every perturbation has its own rotation, a pair is one direct residual evaluation
        # (REG 26, REPROJ 31 + reciprocal, POSE_REG 36 flop); no shared set-up
        fpa = fpl = {1: 31.0, 2: 26.0}.get(inst.residual_type, 36.0)
        fsa = fsl = 0.0
    flops64 = fpa * st["perturb_pairs"] + fpl * st["ladder_pairs"] + fsa * st["perturb_setups"] + fsl * st["ladder_setups"]
    flops32 = fpa * st["perturb_pairs_f32"] + fpl * st["ladder_pairs_f32"]
    flops = flops64 + flops32
    t_min = flops64 / peak64 + flops32 / peak32
    nom32, nom64 = 148 * 128 * 2 * nom_mhz * 1e6, 148 * 64 * 2 * nom_mhz * 1e6
    # the integer work a flop count does not see: one Philox4x32-10 call per perturbation and iteration
    philox_calls = float(st["walker_steps"]) * (P.n_p + 1)
    pairs = st["perturb_pairs"] + st["ladder_pairs"] + st["perturb_pairs_f32"] + st["ladder_pairs_f32"]
    ws = max(1, st["walker_steps"])
    # ALGORITHMIC arithmetic of a launch: eq. (14) as Alg. 3 states it, every perturbation against every constraint
    # (N_P x N pairs per walker-step: shared-R form, 7 flop per pair), plus the ladder pairs and set-ups the
    # first-feasible-rung walk needs (executed counts: data dependent).  The dense kernels execute exactly that (plus the
    # padding of odd runs); the branch-and-bound kernel (N_P <= 32) proves most eq. (14) pairs irrelevant and skips them,
    # so its EXECUTED arithmetic is lower: both fractions are reported, `frac` on the algorithmic count.
    extra32 = 0.0
    if wl.mode != "trans":
        extra32 = max(0.0, fpa * (float(ws) * P.n_p * inst.n - st["perturb_pairs_f32"] - st["perturb_pairs"]))
    flops_alg = flops + extra32
    t_alg = t_min + extra32 / peak32
    roof = {"bound": "alu", "kernel": wl.kernel, "achieved": flops_alg / walk_s / 1e12, "peak": flops_alg / t_alg / 1e12,
            "unit": "TFLOP/s", "frac": t_alg / walk_s,
            "traffic": _traffic(inst.name, wl.mode, wl.precision, wl.W, wl.S, wl.nb),
            "definition": "achieved = algorithmic flops per launch (7 x N_P x N eq. (14) pairs per walker-step + executed ladder "
                          "pairs and set-ups) / kernel time; peak = the same flops / (fp64 flops / DFMA peak + fp32 flops / FFMA "
                          "peak), both peaks measured in this run by closure_alu_peak (register-resident FMA chains)",
            "flops_per_launch": flops_alg,
            # what the kernel actually executed (its own counters; cross-checked against ncu in profiles/): equal to the
            # algorithmic count for the dense kernels, a quarter of it for the branch and bound of config C5
            "executed": {"flops_per_launch": flops, "achieved": flops / walk_s / 1e12, "frac": t_min / walk_s},
            "frac_executed": t_min / walk_s,
            "fp32": {"flops_per_launch": flops32, "achieved": flops32 / walk_s / 1e12, "peak": peak32 / 1e12},
            "fp64": {"flops_per_launch": flops64, "achieved": flops64 / walk_s / 1e12, "peak": peak64 / 1e12},
            # the unit-count peak of SURVEY.md 8(d): 148 SMs x 128 FP32 (64 FP64) lanes x 2 x the maximum SM clock
            "frac_of_nominal": ((flops32 + extra32) / nom32 + flops64 / nom64) / walk_s,
            "peak_nominal": {"fp32": nom32 / 1e12, "fp64": nom64 / 1e12, "sm_mhz": nom_mhz},
            "philox": {"calls_per_launch": philox_calls, "peak_calls_per_s": peak_philox,
                       "note": "Philox4x32-10 calls at the rate of a kernel that does nothing else"},
            "frac_incl_philox": (t_alg + philox_calls / peak_philox) / walk_s,
            "executed_pairs_per_walker_step": pairs / ws,
            "nominal_pairs_per_walker_step": (P.n_p + P.n_p_star * P.n_t) * inst.n,
            "fp64_fallback_steps": st["fallback_steps"] / ws,
            "accepted_steps": st["accepted_steps"] / ws,
            "setup_share_of_warp_cycles": (st["setup_cycles"] / st["total_cycles"]) if st.get("total_cycles") else None}
    return roof, st


def e2e_of(wl: Workload, steps: int) -> dict:
    """End to end through the C ABI with HOST buffers, every step: closure_create + closure_set_init (H2D) +
    closure_run (walk, compaction, count D2H, MEGB with its own D2H) + destroy, for every instance of the batch."""
    torch, B = wl.torch, wl.B
    megb_s, megb_max, d2h, pivots, slowest = [], 0.0, 0, 0, (0.0, 0.0)
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    for k in range(steps):
        for b, (it, s0) in enumerate(zip(wl.insts, wl.S0s)):
            h = B.Closure.closure_create(it)
            h.closure_set_init(s0)
            r = h.closure_run(wl.W, wl.S, WALK_SEED + k + 1000 * b, wl.stream)
            megb_s.append(r["host_seconds"])
            megb_max = max(megb_max, r["max_pivot_seconds"])
            slowest = max(slowest, (r["host_seconds"], r["prepare_seconds"]))
            d2h += r["d2h_bytes"] + 8                    # what closure_megb copied + the 8-byte count
            pivots += r["pivots"]
            h.closure_destroy()
    torch.cuda.synchronize()
    dt = time.perf_counter() - t0
    h2d = sum(it.measurements.nbytes + it.betas.nbytes + s0.nbytes + 256 for it, s0 in zip(wl.insts, wl.S0s))
    return {"value": steps * wl.nb * wl.W * wl.S / dt, "unit": UNIT, "h2d_bytes_per_step": h2d,
            "d2h_bytes_per_step": d2h // steps,
            "d2h_note": "bytes actually copied: 8 (count) + closure_megb_result.d2h_bytes per instance -- clouds of >= 4,096 "
                        "samples stay on the device (16 B per miniball pivot + the fetched support candidates)",
            "buffers": "closure_run's device buffers are cached per process and device: create/destroy in this loop allocates once",
            "per_instance_ms": 1e3 * dt / (steps * wl.nb), "steps": steps,
            "megb_ms_median": 1e3 * statistics.median(megb_s), "megb_ms_max": 1e3 * max(megb_s),
            "megb_pivots_per_instance": pivots / (steps * wl.nb), "megb_slowest_pivot_ms": 1e3 * megb_max,
            "megb_slowest_call": {"ms": 1e3 * slowest[0], "of_which_prepare_ms": 1e3 * slowest[1],
                                  "note": "prepare = embedding pass + cudaMalloc of the per-device cloud buffers when a larger cloud "
                                          "than any before arrives (once per process and size): the source of the rare 20-90 ms calls"}}


def latency_split(wl: Workload, reps: int = 5) -> dict:
    """Per-instance latency by component, mirroring Table IV: create (H2D of the constraint
    table) / set_init (host check of S_0, mean pose, H2D) / sample / compact / D2H of the count / MEGB; wall clock
    with a synchronise after every component, median of `reps` on instance 0."""
    torch, B = wl.torch, wl.B
    it, s0 = wl.insts[0], wl.S0s[0]
    smp = wl.samples[:wl.W]
    flg = wl.flags[:wl.W]
    cmp_ = wl.compacted[:wl.W]
    acc = {k: [] for k in ("create", "set_init", "sample", "compact", "d2h_count", "megb", "destroy", "total")}
    for k in range(reps):
        torch.cuda.synchronize()
        t = [time.perf_counter()]
        h = B.Closure.closure_create(it); t.append(time.perf_counter())
        h.closure_set_init(s0); t.append(time.perf_counter())
        h.closure_sample(wl.W, wl.S, WALK_SEED + k, smp, flg, wl.stream); torch.cuda.synchronize(); t.append(time.perf_counter())
        h.closure_compact(smp, flg, cmp_, wl.count, wl.stream); torch.cuda.synchronize(); t.append(time.perf_counter())
        cnt = int(wl.count.item()); t.append(time.perf_counter())
        if cnt > 0:
            h.closure_megb(cmp_, cnt, wl.stream)
        t.append(time.perf_counter())
        h.closure_destroy(); t.append(time.perf_counter())
        for name, a, b in zip(("create", "set_init", "sample", "compact", "d2h_count", "megb", "destroy"), t[:-1], t[1:]):
            acc[name].append(1e3 * (b - a))
        acc["total"].append(1e3 * (t[-1] - t[0]))
    out = {k: statistics.median(v) for k, v in acc.items()}
    out["note"] = (f"ms, median of {reps}, instance 0: {wl.W} walkers x {wl.S} iterations; host wall clock, "
                   "synchronised after every component")
    return out


def small_scale(B, torch, inst, S0, stream, walkers: int, iterations: int, reps: int = 25) -> dict:
    """The paper's own scale (|S_0| N_W walks, N_I iterations): host buffers in, MEGB out
    through closure_create + closure_set_init + closure_run, and the walker kernel's share by CUDA events."""
    ms = []
    for k in range(reps):
        t1 = time.perf_counter()
        h = B.Closure.closure_create(inst)
        h.closure_set_init(S0)
        h.closure_run(walkers, iterations, WALK_SEED + k, stream)
        h.closure_destroy()
        ms.append(1e3 * (time.perf_counter() - t1))
    h = B.Closure.closure_create(inst)
    h.closure_set_init(S0)
    dev = torch.device("cuda", torch.cuda.current_device())
    smp = torch.empty((walkers, 12), dtype=torch.float64, device=dev)
    flg = torch.empty((walkers,), dtype=torch.uint8, device=dev)
    kms = []
    for k in range(12):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        h.closure_sample(walkers, iterations, WALK_SEED + k, smp, flg, stream)
        e1.record(stream)
        torch.cuda.synchronize()
        kms.append(e0.elapsed_time(e1))
    h.closure_destroy()
    e2e, kern = statistics.median(ms[5:]), statistics.median(kms[2:])
    return {"walkers": walkers, "iterations": iterations, "e2e_ms": e2e, "walker_kernel_ms": kern,
            "walker_kernel_share": kern / e2e, "walker_steps_per_sec_e2e": walkers * iterations / (e2e * 1e-3)}


def run_cuda(args) -> None:
    import torch
    import torch.distributed as dist
    from paper_2403_09990_b200 import binding as B
    from paper_2403_09990_b200 import sharding

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

    dev = torch.device("cuda", local)
    flush = torch.empty((256 << 20,), dtype=torch.uint8, device=dev)      # > 126 MB L2

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    if args.scaling == "strong" and world > 1:
        out = run_strong(args, B, torch, dist, sharding, rank, world, local, flush, barrier)
        dist.barrier()
        dist.destroy_process_group()
        if out is not None:
            print(json.dumps(out))
        return

    # Weak scaling: every rank walks W walkers per instance with its own
    # walker-id range [rank*W, (rank+1)*W); walkers are independent, no collective
    # sits on the data path.
    inst0, _ = _workload(args.config)
    W0 = int(args.walkers or inst0.num_walkers)
    wl = Workload(B, torch, args.config, args.mode, args.precision, begin=rank * W0, walkers=args.walkers,
                  iterations=args.iterations)
    inst, S0, P = wl.inst, wl.S0, wl.inst.params
    W, S, nb = wl.W, wl.S, wl.nb
    stream = wl.stream

    peak64, _ = B.closure_alu_peak(64)
    peak32, _ = B.closure_alu_peak(32)
    peak_philox, _ = B.closure_alu_peak(4)          # Philox4x32-10 calls per second
    clocks = ClockSampler(local)
    # warm-up outside the clock sample, then the timed region
    for w in range(args.warmup):
        wl.step(WALK_SEED + 100 + w)
        flush.fill_(w)
    barrier()
    clocks.start()
    total_ms, walk_ms, comp_ms = timed_steps(wl, args.steps, 0, flush, barrier)
    clk = clocks.stop()
    if world > 1:
        tt = torch.tensor([total_ms], dtype=torch.float64, device=dev)
        dist.all_reduce(tt, op=dist.ReduceOp.MAX)
        total_ms = float(tt.item())
    units = float(world) * nb * W * S * args.steps
    value = units / (total_ms * 1e-3)

    out, peaks = None, None
    if rank == 0:
        nom_mhz = float(clk.get("sm_max_mhz") or 1965.0)
        peaks = {"f64": peak64, "f32": peak32, "philox": peak_philox, "nom_mhz": nom_mhz}
        walk_s = statistics.mean(walk_ms) * 1e-3
        roof, st = roofline_of(wl, walk_s, peaks)
        nominal_pairs = (P.n_p + P.n_p_star * P.n_t) * inst.n
        n_cnt = int(wl.count.item())
        comp_bytes = nb * W * 1 + n_cnt * 96 * 2
        comp_s = statistics.mean(comp_ms) * 1e-3
        mp = {}
        try:
            mp = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
        except OSError:
            pass
        hbm_peak = float(mp.get("hbm_gbs", 6650.0))

        e2e = e2e_of(wl, max(1, min(args.steps, 2 if nb > 1 else 3)))
        split = latency_split(wl)

        # Step I on the device (not part of the timed step): trials -> compaction -> S_0 for
        # 1,000 trials end to end, and the trial kernel alone at the 100,000 trials of the paper's pure-RANSAG
        # comparison.  Ex.1: P3P trials; Ex.2: Arun; Ex.3: convex combinations.
        hs1 = B.Closure.closure_create(wl.insts[0])
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
            import oracle
            Wc = min(W, 16384)
            P64 = copy.copy(wl.insts[0].params)
            P64.precision = 64
            h64 = B.Closure.closure_create(wl.insts[0], P64)
            h64.closure_set_init(wl.S0s[0])
            s32, f32_, t32 = wl.handles[0].closure_sample(Wc, S, WALK_SEED, trace=True)
            s64, f64_, t64 = h64.closure_sample(Wc, S, WALK_SEED, trace=True)
            same = (t32 == t64).all(dim=1)
            c32, n32 = wl.handles[0].closure_compact(s32, f32_)
            r32 = wl.handles[0].closure_megb(c32, int(n32.item()))
            c64, n64 = h64.closure_compact(s64, f64_)
            r64 = h64.closure_megb(c64, int(n64.item()))
            worst = min(oracle.margin(wl.insts[0], s[:9], s[9:]) for s in s32[::max(1, Wc // 512)].cpu().numpy())
            fp32_report = {"walkers_compared": Wc, "iterations": S,
                           "walkers_with_identical_decisions": float(same.float().mean().item()),
                           "max_abs_sample_difference_among_those": float((s32[same] - s64[same]).abs().max().item())
                           if bool(same.any()) else None,
                           "worst_emitted_sample_margin": worst,
                           "rot_radius_rel_diff": abs(r32["rot_radius"] - r64["rot_radius"]) / r64["rot_radius"],
                           "trans_radius_rel_diff": abs(r32["trans_radius"] - r64["trans_radius"]) / r64["trans_radius"]}
            h64.closure_destroy()
            del s32, s64, t32, t64

        # the compaction kernel alone at BASELINE config 5's size (4,194,304 walkers): the size at which it is
        # HBM-bound rather than launch-bound; every sample kept, and every second one
        nbig = 4194304
        if nb * W == nbig:
            big_s, big_o = wl.samples, wl.compacted
        else:
            big_s = torch.empty((nbig, 12), dtype=torch.float64, device=dev).fill_(1.0)
            big_o = torch.empty_like(big_s)
        comp_big = {}
        for label, big_f in (("all_kept", torch.ones((nbig,), dtype=torch.uint8, device=dev)),
                             ("half_kept", (torch.arange(nbig, device=dev) % 2).to(torch.uint8))):
            big_ms = []
            for k in range(7):
                flush.fill_(k)
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record(stream)
                wl.handles[0].closure_compact(big_s, big_f, big_o, wl.count, stream)
                e1.record(stream)
                torch.cuda.synchronize()
                if k >= 2:
                    big_ms.append(e0.elapsed_time(e1))
            big_bytes = nbig * 1 + int(wl.count.item()) * 96 * 2
            big_gbs = big_bytes / (statistics.mean(big_ms) * 1e-3) / 1e9
            comp_big[label] = {"achieved": big_gbs, "frac": big_gbs / hbm_peak, "bytes_per_launch": big_bytes,
                               "ms": statistics.mean(big_ms)}
        # context for the fraction above: a plain device-to-device copy of the same payload (cudaMemcpyAsync through torch),
        # timed the same way -- what a kernel-free copy of 402.7 MB reaches of the measured peak on this box
        copy_ms = []
        for k in range(7):
            flush.fill_(k)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            big_o.copy_(big_s, non_blocking=True)
            e1.record(stream)
            torch.cuda.synchronize()
            if k >= 2:
                copy_ms.append(e0.elapsed_time(e1))
        copy_gbs = nbig * 96 * 2 / (statistics.mean(copy_ms) * 1e-3) / 1e9
        comp_big["memcpy_same_payload"] = {"achieved": copy_gbs, "frac": copy_gbs / hbm_peak, "bytes_per_launch": nbig * 96 * 2,
                                           "ms": statistics.mean(copy_ms)}
        big_s = big_o = None

        out = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": total_ms / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None,
            "dtype": DTYPE if args.precision == 64 else "f32 decisions (uncertified), f64 poses", "data": "synthetic",
            "config": _config_dict(inst, W, S, nb, "walker ranges per rank, no collective"),
            "constraint_evals_per_sec_nominal": value * nominal_pairs,
            "constraint_evals_per_sec_executed": (st["perturb_pairs"] + st["ladder_pairs"] + st["perturb_pairs_f32"]
                                                  + st["ladder_pairs_f32"]) / walk_s * world,
            "latency_ms": {"walker_kernel": statistics.mean(walk_ms), "compaction_kernel": statistics.mean(comp_ms),
                           "megb": e2e["megb_ms_median"], "megb_max": e2e["megb_ms_max"],
                           "e2e_per_instance": e2e["per_instance_ms"], "per_instance_split": split},
            "boundary_fraction": n_cnt / float(nb * W),
            "roofline": roof,
            "roofline_compaction": {"bound": "hbm", "kernel": "compact_kernel", "achieved": comp_bytes / comp_s / 1e9,
                                    "peak": hbm_peak, "unit": "GB/s", "frac": comp_bytes / comp_s / 1e9 / hbm_peak,
                                    "bytes_per_launch": comp_bytes, "peak_source": "MEASURED_PEAKS.json hbm_gbs"
                                    if mp else "fallback 6650",
                                    "at_4194304_walkers": comp_big["all_kept"],
                                    "at_4194304_walkers_half_kept": comp_big["half_kept"],
                                    "memcpy_same_payload": comp_big["memcpy_same_payload"]},
            "e2e": e2e,
            "gpu_launches": args.steps * (-(-nb // 96) + 1),     # walker launch(es) + compaction kernel per step
            "clocks": clk,
        }
        if fp32_report is not None:
            out["fp32_mode"] = fp32_report
        out["step1"] = step1
    wl.destroy()

    if rank == 0 and world == 1 and not args.no_per_config:
        out["per_config"] = per_config_block(B, torch, args, peaks, flush, barrier)
        out["moving_regime"] = moving_regime_block(B, torch, args, peaks, flush, barrier, out["per_config"])
    if rank == 0 and not args.no_cpu_baseline and world == 1:
        out["cpu_baseline"] = cpu_baseline(inst, S0)
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()
    if out is not None:
        print(json.dumps(out))


def per_config_block(B, torch, args, peaks, flush, barrier) -> list:
    """One short measurement of every other BASELINE config at full size (3 warm-up + 2 timed steps each), so that all
    five configs are observed by the same run; same timing rules as the headline."""
    rows = []
    for cfg, mode in PER_CONFIG:
        if cfg == args.config and mode == args.mode and not args.walkers and not args.iterations:
            continue
        wl = Workload(B, torch, cfg, mode, 64)
        total_ms, walk_ms, comp_ms = timed_steps(wl, 2, 3, flush, barrier)
        walk_s = statistics.mean(walk_ms) * 1e-3
        roof, st = roofline_of(wl, walk_s, peaks)
        e2e = e2e_of(wl, 1)
        P = wl.inst.params
        v = wl.nb * wl.W * wl.S * 2 / (total_ms * 1e-3)
        rows.append({"workload": wl.inst.name, "mode": mode, "N": wl.inst.n, "walkers": wl.W, "iterations": wl.S,
                     "instances": wl.nb, "params": _params_dict(P), "steps": 2, "warmup": 3,
                     "value": v, "unit": UNIT, "ms_per_step": total_ms / 2,
                     "walker_kernel_ms": statistics.mean(walk_ms), "compaction_kernel_ms": statistics.mean(comp_ms),
                     "constraint_evals_per_sec_nominal": v * (P.n_p + P.n_p_star * P.n_t) * wl.inst.n,
                     "boundary_fraction": int(wl.count.item()) / float(wl.nb * wl.W),
                     "roofline": {k: roof[k] for k in ("kernel", "achieved", "peak", "unit", "frac", "frac_of_nominal",
                                                       "frac_incl_philox", "frac_executed", "executed_pairs_per_walker_step",
                                                       "fp64_fallback_steps", "accepted_steps", "traffic")},
                     "e2e": {k: e2e[k] for k in ("value", "unit", "per_instance_ms", "h2d_bytes_per_step",
                                                 "d2h_bytes_per_step", "megb_ms_median")}})
        wl.destroy()
    return rows


def moving_regime_block(B, torch, args, peaks, flush, barrier, per_config) -> dict:
    """The regime the paper runs: N_I = 5 and 20 iterations, where most iterations move the walker
    and the set-up that follows a move is paid every time.  65,536 walkers at C2 and C3; the stuck-regime number of
    the same config (1,000 iterations) is repeated beside it.  Also the paper's own batch sizes end to end:
    |S_0| N_W = 200 walks x N_I = 5 (CLOSURE) and 2,000 x 10 (CLOSURE++)."""
    rows = []
    stuck = {(r["workload"], r["mode"]): r["value"] for r in per_config}
    for cfg in (2, 3):
        for n_i in (5, 20):
            wl = Workload(B, torch, cfg, "rot", 64, walkers=65536, iterations=n_i)
            total_ms, walk_ms, comp_ms = timed_steps(wl, 5, 3, flush, barrier)
            walk_s = statistics.mean(walk_ms) * 1e-3
            roof, st = roofline_of(wl, walk_s, peaks)
            ref = stuck.get((wl.inst.name, "rot"))
            rows.append({"workload": wl.inst.name, "walkers": wl.W, "iterations": n_i,
                         "value": wl.W * wl.S * 5 / (total_ms * 1e-3), "unit": UNIT,
                         "walker_kernel_ms": statistics.mean(walk_ms), "ms_per_step": total_ms / 5,
                         "walker_steps_per_sec_kernel_only": wl.W * wl.S / walk_s,
                         "accepted_steps": roof["accepted_steps"],
                         "setup_share_of_warp_cycles": roof["setup_share_of_warp_cycles"],
                         "roofline_frac": roof["frac"],
                         "executed_pairs_per_walker_step": roof["executed_pairs_per_walker_step"],
                         "stuck_regime_value": ref,
                         "kernel_only_vs_stuck_regime": (wl.W * wl.S / walk_s) / ref if ref else None})
            wl.destroy()
    paper = []
    for cfg in (2, 3):
        inst, S0 = _workload(cfg)
        for walkers, n_i in ((200, 5), (2000, 10)):
            r = small_scale(B, torch, inst, S0, torch.cuda.current_stream(), walkers, n_i)
            r["workload"] = inst.name
            paper.append(r)
    return {"at_65536_walkers": rows, "paper_scale_end_to_end": paper,
            "context": "the paper reports 84-92 ms (CLOSURE) and 0.62-1.20 s (CLOSURE++) for the walk per instance on an "
                       "RTX 3090 with CuPy (Table IV, PAPER.md:491-496): another machine, context only"}


def run_strong(args, B, torch, dist, sharding, rank, world, local, flush, barrier):
    """--scaling strong at N > 1 ranks: ONE job split over the ranks.  A single instance is
    split by walker ranges (closure_sample_range), every rank compacts its own samples, the compacted clouds are
    gathered unpadded on rank 0 (counts first, then point-to-point payloads into a buffer sized from the counts)
    and rank 0 runs closure_megb on the merged cloud; a batch of instances (C5) is split by whole instances and
    needs no exchange.  Philox keys make walker w placement-independent, so the merged cloud and its MEGB equal
    the one-GPU run bit for bit (tests/test_multirank_gloo.py drives the same sharding.strong_step on gloo)."""
    inst, S0 = _workload(args.config)
    if args.mode == "trans":
        inst.params.mode = I.MODE_TRANS
    W = int(args.walkers or inst.num_walkers)
    S = int(args.iterations or inst.num_steps)
    nb = inst.batch
    dev = torch.device("cuda", local)
    stream = torch.cuda.current_stream()
    if nb > 1:
        mine = list(range(rank, nb, world))                # whole instances, round-robin
        insts = [I.make_instance(args.config, b) for b in mine]
        S0s = [I.make_init_poses(it, 128) for it in insts]
        handles = []
        for it, s0 in zip(insts, S0s):
            h = B.Closure.closure_create(it)
            h.closure_set_init(s0)
            handles.append(h)
        smp = torch.empty((max(len(mine), 1), W, 12), dtype=torch.float64, device=dev)
        flg = torch.empty((max(len(mine), 1), W), dtype=torch.uint8, device=dev)
        cmp_ = torch.empty((max(len(mine), 1) * W, 12), dtype=torch.float64, device=dev)
        cnt = torch.zeros((1,), dtype=torch.int64, device=dev)

        def step(seed):
            if mine:
                B.closure_sample_batch(handles, W, S, [seed + 1000 * b for b in mine], smp, flg, stream)
                handles[0].closure_compact(smp.view(-1, 12), flg.view(-1), cmp_, cnt, stream)
            return None
    else:
        h = B.Closure.closure_create(inst)
        h.closure_set_init(S0)
        handles = [h]
        _, mine_w = sharding.walker_range(rank, world, W)
        smp = torch.empty((max(mine_w, 1), 12), dtype=torch.float64, device=dev)
        flg = torch.empty((max(mine_w, 1),), dtype=torch.uint8, device=dev)
        cmp_ = torch.empty((max(mine_w, 1), 12), dtype=torch.float64, device=dev)
        cnt = torch.zeros((1,), dtype=torch.int64, device=dev)

        def step(seed):
            return sharding.strong_step(
                sample=lambda b, n: h.closure_sample(n, S, seed, smp[:n], flg[:n], stream, walker_begin=b),
                compact=lambda s, f: h.closure_compact(s, f, cmp_[:s.shape[0]], cnt, stream),
                megb=lambda cloud, c: h.closure_megb(cloud, c, stream),
                num_walkers=W, rank=rank, world=world, device=dev)

    for w in range(args.warmup):
        step(WALK_SEED + 100 + w)
        flush.fill_(w)
    barrier()
    clocks = ClockSampler(local)
    clocks.start()
    t0, t1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    t0.record(stream)
    res = None
    for k in range(args.steps):
        res = step(WALK_SEED + k)
        flush.fill_(k)
    t1.record(stream)
    barrier()
    clk = clocks.stop()
    tt = torch.tensor([t0.elapsed_time(t1)], dtype=torch.float64, device=dev)
    dist.all_reduce(tt, op=dist.ReduceOp.MAX)
    total_ms = float(tt.item())
    for hh in handles:
        hh.closure_destroy()
    if rank != 0:
        return None
    value = nb * W * S * args.steps / (total_ms * 1e-3)
    out = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world,
           "steps": args.steps, "warmup": args.warmup, "ms_per_step": total_ms / args.steps, "higher_is_better": True,
           "scaling": "strong", "vs_baseline": None, "dtype": DTYPE, "data": "synthetic",
           "config": _config_dict(inst, W, S, nb, "whole instances per rank, no exchange" if nb > 1 else
                                  "walker ranges of one instance per rank; compacted samples gathered unpadded on rank 0 "
                                  "(NCCL point-to-point), MEGB on rank 0, inside the timed step"),
           "gpu_launches": args.steps * 2, "clocks": clk,
           "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0,
                   "note": "strong-scaling mode times the device-resident step; the host-buffer end-to-end number is "
                           "the one-GPU line's"}}
    if res is not None and res.get("count"):
        out["megb"] = {"rot_radius": res["rot_radius"], "trans_radius": res["trans_radius"], "count": res["count"]}
    return out


def main() -> None:
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="cuda", choices=["cuda", "reference"])
    ap.add_argument("--config", type=int, default=5,
                    help="BASELINE.json config 1..5 (default 5 = configs[4], the largest single-GPU workload)")
    ap.add_argument("--iterations", type=int, default=0, help="override the config's iterations per walker (N_I)")
    ap.add_argument("--walkers", type=int, default=0, help="override the config's walkers per instance")
    ap.add_argument("--scaling", default="weak", choices=["weak", "strong"],
                    help="N > 1 ranks: weak = every rank runs the whole workload on its own walker ids (default); "
                         "strong = one workload split over the ranks, with the gather + MEGB on rank 0")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-per-config", action="store_true", help="skip the per_config and moving_regime blocks")
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
