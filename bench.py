#!/usr/bin/env python
"""bench.py — BASELINE.json's metric on BASELINE.json's headline config, through the C ABI of libens.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]

Metric: Hermite FP64 system-steps/s on config 1 (131072 systems x 3 bodies, dt = 0.01, 10^4 steps per launch, close
approach and ejection monitors armed).  One bench "step" is one pass of the hot path over the whole ensemble:
ens_set_state (AoS -> SoA, inputs already resident in HBM) -> ens_integrate(HERMITE, 10^4 steps: load, 3 x
acc+jerk, predictor, 2 x corrector, monitors, retire, store) -> ens_energy.  `value` = system-steps actually taken by
all GPUs / seconds per step.  `e2e` is the same pass through HOST buffers (pinned), host<->device copies inside the
timed region.  Every other step-loop kernel of the library (configs 2-4 at full size, the adaptive / 2-evaluation /
Cash-Karp / merged-MVS kernels, the paper's own workload shapes, every n_body) rides along under `other_workloads`,
`paper_shapes` and `all_n`, each with its algorithmic work and the fraction of the FP64 roofline it reaches.

N > 1 (torchrun): every rank integrates its own config-1 ensemble (different system indices, no data-path
collective: systems are independent) -> weak scaling; time = max over ranks.
`--impl reference` times the CPU oracle (rank 0 only) on a bounded sample of the same workload.
"""
from __future__ import annotations

import argparse
import json
import os
import re
import statistics
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from paper_1208_1157_b200 import workloads as W  # noqa: E402

METRIC = "hermite_fp64_system_steps_per_sec_131072x3"
UNIT = "system-steps/s"
CFG = 1

# ---------------------------------------------------------------------------------------------------------------
# Algorithmic FP64 work of one system-step of every step-loop kernel (each unordered pair once
# per evaluation; FMA = 1 instruction = 2 flops, add / mul = 1).  Derived from the method, cross-checked against
# sm__sass_thread_inst_executed_op_{dfma,dmul,dadd}_pred_on of the ncu summaries under profiles/ (r2_opcounts.md).
# ---------------------------------------------------------------------------------------------------------------
PAIR_INSTR, PAIR_FLOPS = 38, 60           # one pair acc+jerk evaluation
COMP_INSTR, COMP_FLOPS = 17, 34           # Hermite predictor + 2 correctors, per body component
BODY_MON_INSTR, BODY_MON_FLOPS = 0, 0     # monitors: the step loops test high words on the integer ALU (no FP64 work)
ACC_PAIR_INSTR, ACC_PAIR_FLOPS = 21, 32   # one pair, acceleration only (Cash-Karp stages, MVS planet pairs)
R2_PAIR_INSTR, R2_PAIR_FLOPS = 6, 8       # one pair separation, positions only (monitor of the 2-evaluation Hermite)


def _pairs(n):
    return n * (n - 1) // 2


def hermite_work(n_body: int):
    """3 evaluations per step (R6): 3 P 38 + 3 N 17 + 1 (the time update); the monitors cost no FP64 instruction."""
    p = _pairs(n_body)
    return (3 * p * PAIR_INSTR + 3 * n_body * COMP_INSTR + n_body * BODY_MON_INSTR + 1,
            3 * p * PAIR_FLOPS + 3 * n_body * COMP_FLOPS + n_body * BODY_MON_FLOPS + 1)


def hermite_carry_work(n_body: int):
    """Alg. 2 as printed: 2 evaluations per step + the positions-only separation pass of its close-approach monitor."""
    p = _pairs(n_body)
    return (2 * p * PAIR_INSTR + p * R2_PAIR_INSTR + 3 * n_body * COMP_INSTR + n_body * BODY_MON_INSTR + 1,
            2 * p * PAIR_FLOPS + p * R2_PAIR_FLOPS + 3 * n_body * COMP_FLOPS + n_body * BODY_MON_FLOPS + 1)


def hermite_adaptive_work(n_body: int):
    """Hermite + Eq. 5 (|a|^2, |j|^2, reciprocal per body; rsqrt) + the step-size powers rebuilt from the per-system h."""
    i, f = hermite_work(n_body)
    return i + 12 * n_body + 26, f + 17 * n_body + 32


def rkck_work(n_body: int):
    """6 acceleration evaluations + 25 DFMA per coordinate (stage positions, fifth-order solution)."""
    p = _pairs(n_body)
    return (6 * p * ACC_PAIR_INSTR + 3 * n_body * 25 + n_body * BODY_MON_INSTR + 1,
            6 * p * ACC_PAIR_FLOPS + 3 * n_body * 50 + n_body * BODY_MON_FLOPS + 1)


def rkck_adaptive_work(n_body: int):
    """Per ACCEPTED step (rejected trials are overhead, not work): the fixed-step work with the powers of h applied per
    system (44 instead of 25 per coordinate incl. the error sums), the scale norms and the control."""
    p = _pairs(n_body)
    return (6 * p * ACC_PAIR_INSTR + 3 * n_body * 44 + n_body * (BODY_MON_INSTR + 8) + 30,
            6 * p * ACC_PAIR_FLOPS + 3 * n_body * 76 + n_body * (BODY_MON_FLOPS + 12) + 45)


def mvs_work(n_body: int, merged: bool = False):
    """Per planet: universal-variable Kepler drift 111 (setup 17, series start 18, one 7-term Stumpff evaluation +
    Chebyshev step 39 with its tests on the integer ALU, Taylor finish + f, g functions 37), drifts / kicks / momentum sum 15 (merged: 12); per system 16
    (merged: 13); planet pairs 21 each.  The monitors cost no FP64 instruction (high words, integer ALU)."""
    pl = n_body - 1
    pp = _pairs(pl)
    per_planet_i, per_planet_f = (111 + 12, 172 + 20) if merged else (111 + 15, 172 + 24)
    per_sys_i, per_sys_f = (13, 19) if merged else (16, 22)
    return pl * per_planet_i + per_sys_i + pp * ACC_PAIR_INSTR, pl * per_planet_f + per_sys_f + pp * ACC_PAIR_FLOPS


WORK = {
    "hermite": hermite_work, "hermite_carry": hermite_carry_work, "hermite_adaptive": hermite_adaptive_work,
    "rkck": rkck_work, "rkck_adaptive": rkck_adaptive_work, "mvs": mvs_work,
    "mvs_merged": lambda n: mvs_work(n, merged=True),
}

# FP64 peak of a B200: 148 SMs x 64 FP64 lanes x 1 FMA/clk x max SM clock.
FP64_LANES_PER_SM = 64


def nominal_fp64_peak(sm_count: int, sm_max_mhz: float):
    lane_inst = sm_count * FP64_LANES_PER_SM * sm_max_mhz * 1e6
    return lane_inst, 2.0 * lane_inst / 1e12  # lane-instr/s, TFLOP/s


def profile_traffic(path: str):
    """dram__bytes_read.sum + dram__bytes_write.sum of one launch, read from a committed ncu summary (text, under
    profiles/).  None when the file or the metrics are missing: the line then carries no traffic figure at all."""
    try:
        text = open(path).read()
    except OSError:
        return None
    tot, found = 0.0, 0
    for key in ("dram__bytes_read.sum", "dram__bytes_write.sum"):
        m = re.search(r"^" + re.escape(key) + r"\s+([0-9.eE+-]+)\s+(\S+)", text, re.M)
        if not m:
            continue
        scale = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9}.get(m.group(2))
        if scale is None:
            continue
        tot += float(m.group(1)) * scale
        found += 1
    return tot if found == 2 else None


class ClockSampler:
    """nvidia-smi clocks and throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.rows, self.proc, self.index = [], None, index

    def __enter__(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "100"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thr = threading.Thread(target=self._read, daemon=True)
            self.thr.start()
        except OSError:
            self.proc = None
        return self

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def __exit__(self, *exc):
        if self.proc:
            self.proc.terminate()
            try:
                self.proc.wait(timeout=5)
            except Exception:
                self.proc.kill()
            self.thr.join(timeout=2)

    def summary(self):
        sm, mx, pw, reasons = [], [], [], set()
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1])); pw.append(float(r[2]))
            except (ValueError, IndexError):
                continue
            for name, val in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[3:7]):
                if val.lower().startswith("active"):
                    reasons.add(name)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        # "under load": samples in the upper half of the power range
        lo, hi = min(pw), max(pw)
        load = [c for c, p in zip(sm, pw) if p >= lo + 0.5 * (hi - lo)] or sm
        return {"sm_mhz": statistics.median(load), "sm_max_mhz": max(mx), "power_w_max": hi,
                "reasons": sorted(reasons), "samples": len(sm)}


# ---------------------------------------------------------------------------------------------------------------
# The oracle legs.  ONE sample definition serves both `cpu_baseline` and `--impl reference`: the first
# SAMPLE_PER_CORE x cores systems of config 1 for the full 10^4 steps, system-per-thread OpenMP (the paper's CPU
# scheme), the oracle exactly as it stands.
# ---------------------------------------------------------------------------------------------------------------
SAMPLE_PER_CORE = 64


def oracle_sample():
    import oracle
    c = W.CONFIGS[CFG]
    cores = oracle.host_cores()
    n = SAMPLE_PER_CORE * cores
    pos, vel, mass = W.generate(CFG, n_sys=n)

    def run():
        r = oracle.integrate(oracle.HERMITE, pos, vel, mass, dt=c.dt, max_steps=c.steps, r_close=c.r_close,
                             r_eject=c.r_eject, nthreads=cores)
        return int(r["nsteps"].sum())

    desc = f"first {n} systems of config {CFG} x {c.steps} steps per pass (system-per-thread OpenMP, {cores} threads)"
    return run, cores, desc


def cpu_baseline(budget_s: float = 12.0):
    """The oracle on this box's host cores: passes over the sample until ~budget_s of wall time (at least 2)."""
    run, cores, desc = oracle_sample()
    taken, passes, t0 = 0, 0, time.perf_counter()
    while passes < 2 or (time.perf_counter() - t0 < budget_s and passes < 64):
        taken += run()
        passes += 1
    dt = time.perf_counter() - t0
    return {"value": taken / dt, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc,
            "passes": passes, "wall_s": dt,
            "note": "the correctness oracle as it stands (plain loops, -O2, no FMA contraction): a reported baseline, not a tuned CPU code"}


def run_reference(args):
    """--impl reference: the CPU oracle (rank 0 only), each bench step one pass over the same sample."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    c = W.CONFIGS[CFG]
    run, cores, desc = oracle_sample()
    for _ in range(args.warmup):
        run()
    taken, t0 = 0, time.perf_counter()
    for _ in range(args.steps):
        taken += run()
    dt = time.perf_counter() - t0
    value = taken / dt
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": dt / args.steps * 1e3, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": W.CONFIGS[CFG].name, "integrator": "hermite", "dt": c.dt, "sample": desc},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)
    return 0


# ---------------------------------------------------------------------------------------------------------------
# One step-loop kernel on one ensemble: kernel time (the library's own CUDA events around the launch), system-steps
# actually taken, and the fraction of the FP64 roofline its algorithmic work amounts to.
# ---------------------------------------------------------------------------------------------------------------
def time_kernel(ens, torch, stream, kind, integ, arrays, n_body, dt, steps, peak_inst, peak_tf, t_end=float("inf"),
                monitors=(0.0, float("inf")), rk_eps=None, reps=3, event_timed=False):
    n_sys = arrays[0].shape[0]
    d = [torch.from_numpy(x).cuda() if isinstance(x, np.ndarray) else x for x in arrays]
    e = ens.Ensemble(n_sys, n_body)
    try:
        e.set_monitors(*monitors)
        if rk_eps:
            e.set_rk_tolerance(rk_eps)
        ms = []
        for _ in range(reps):
            e.set_state(*d, stream=stream)
            if event_timed:  # kernels with a pre-pass (hand-out order): time the whole C-ABI call
                a0, a1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                a0.record(stream)
                e.integrate(integ, dt, steps, t_end=t_end, stream=stream)
                a1.record(stream)
                a1.synchronize()
                ms.append(a0.elapsed_time(a1))
            else:
                e.integrate(integ, dt, steps, t_end=t_end, stream=stream)
                ms.append(e.last_kernel_ms())
        st = e.get_state(stream=stream)
        info = e.info()
        t = min(ms[1:]) if len(ms) > 1 else ms[0]
        taken = int(st["nsteps"].sum())
        instr, flops = WORK[kind](n_body)
        rate = taken / (t * 1e-3)
        out = {"value": rate, "unit": UNIT, "kernel_ms": t, "n_sys": n_sys, "n_body": n_body, "steps_taken": taken,
               "regs": info["regs"], "stack_bytes": info["stack_bytes"], "blocks_per_sm": info["blocks_per_sm"],
               "lanes_per_system": info["lanes_per_system"], "bodies_per_lane": info["bodies_per_lane"],
               "algorithmic_fp64_instr_per_system_step": instr, "algorithmic_flops_per_system_step": flops,
               "issue_frac_nominal": rate * instr / peak_inst, "frac": rate * flops / 1e12 / peak_tf}
        if info["sliced"]:
            out["grid"] = "time-sliced persistent"
        stopped = int((st["status"] >= 3).sum())
        if stopped:
            out["systems_stopped_by_monitors"] = stopped
        if kind == "rkck_adaptive":
            out["rejected_trial_steps"] = int(e.get_rejected(stream=stream).sum())
        return out
    finally:
        e.close()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=1, choices=[0, 1, 2, 3],
                    help="Hermite workload (BASELINE.json configs index); 1 is the metric's, the others are for profiling")
    ap.add_argument("--no-cpu-baseline", action="store_true", help="skip the oracle timing leg (profiling runs)")
    ap.add_argument("--no-extras", action="store_true", help="skip the e2e / other-kernel / HBM legs (profiling runs)")
    ap.add_argument("--n-sys", type=int, default=None,
                    help="profiling runs: another ensemble size of the same workload (e.g. 18944 = one warp per SM "
                         "sub-partition at n_body = 3); the line says so and is not the metric")
    ap.add_argument("--only", default=None,
                    help="profiling runs: launch just this entry of other_workloads (e.g. mvs_131072x4) a few times and exit")
    args = ap.parse_args()
    global CFG, METRIC
    if args.config != CFG:
        CFG = args.config
        METRIC = "hermite_fp64_system_steps_per_sec_" + W.CONFIGS[CFG].name.split("_", 1)[1]
    if args.impl == "reference":
        return run_reference(args)
    if args.warmup < 3:
        print(f"bench.py: --warmup {args.warmup} is below the 3 warm-up steps a valid timing needs; the number is for "
              "profiling only", file=sys.stderr)

    import torch
    import torch.distributed as dist
    from paper_1208_1157_b200 import ens

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device and no CPU fallback (use --impl reference for the oracle)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    props = torch.cuda.get_device_properties(local)
    stream = torch.cuda.Stream()
    c = W.CONFIGS[CFG]
    n_sys, n_body = c.n_sys, c.n_body
    if args.n_sys:
        n_sys = int(args.n_sys)
        print(f"bench.py: --n-sys {n_sys}: not the metric's ensemble ({c.n_sys}); the number is for profiling only", file=sys.stderr)

    # the other step-loop kernels (kernel time only; none of them the metric).  name -> arguments of time_kernel
    def others_table():
        c1, c2, c3, c4 = (W.CONFIGS[k] for k in (1, 2, 3, 4))
        mon = lambda ck: (ck.r_close, ck.r_eject)
        gen = lambda k: W.generate(k, offset=rank * W.CONFIGS[k].n_sys)
        return {
            c2.name: lambda: ("hermite", ens.HERMITE, gen(2), c2.n_body, c2.dt, c2.steps, dict(monitors=mon(c2))),
            c3.name: lambda: ("hermite", ens.HERMITE, gen(3), c3.n_body, c3.dt, c3.steps, dict(monitors=mon(c3))),
            c4.name: lambda: ("mvs", ens.MVS, gen(4), c4.n_body, c4.dt, c4.steps, dict(monitors=mon(c4))),
            "mvs_merged_131072x4": lambda: ("mvs_merged", ens.MVS_MERGED, gen(4), c4.n_body, c4.dt, c4.steps, dict(monitors=mon(c4))),
            "hermite_carry_131072x3": lambda: ("hermite_carry", ens.HERMITE_CARRY, gen(1), 3, c1.dt, c1.steps, dict(monitors=mon(c1))),
            "rkck_131072x3": lambda: ("rkck", ens.RKCK, gen(1), 3, c1.dt, c1.steps, dict(monitors=mon(c1))),
            # adaptive kernels on the metric's own systems to t = 20: tau = 0.017; eps = 1e-9 (R-RK2')
            "hermite_adaptive_131072x3": lambda: ("hermite_adaptive", ens.HERMITE_ADAPTIVE, gen(1), 3, 0.017, 10**9,
                                                  dict(monitors=mon(c1), t_end=20.0, event_timed=True)),
            "rkck_adaptive_131072x3": lambda: ("rkck_adaptive", ens.RKCK_ADAPTIVE, gen(1), 3, 0.02, 10**9,
                                               dict(monitors=mon(c1), t_end=20.0, rk_eps=1e-9, event_timed=True)),
        }

    peak_inst, peak_tf = nominal_fp64_peak(props.multi_processor_count, 1965.0)

    if args.only:  # one kernel, a few launches, for ncu
        kind, integ, arrays, nb, dt, steps, kw = others_table()[args.only]()
        with torch.cuda.stream(stream):
            r = time_kernel(ens, torch, stream, kind, integ, arrays, nb, dt, steps, peak_inst, peak_tf, reps=max(1, args.steps), **kw)
        print(json.dumps({"only": args.only, **r}), flush=True)
        return 0

    # each rank owns its own range of system indices of the same seeded generator (weak scaling, no exchange)
    from paper_1208_1157_b200 import shard
    lo, hi = shard.weak_range(n_sys, rank)
    pos, vel, mass = W.generate(CFG, n_sys=hi - lo, offset=lo)
    d_pos, d_vel, d_mass = (torch.from_numpy(x).cuda() for x in (pos, vel, mass))
    h_pos, h_vel, h_mass = (torch.from_numpy(x).pin_memory() for x in (pos, vel, mass))
    flush = torch.empty(512 * 1024 * 1024 // 4, dtype=torch.int32, device="cuda")  # 512 MB > 126 MB L2
    e = ens.Ensemble(n_sys, n_body)
    e.set_monitors(c.r_close, c.r_eject)
    e.reserve_host_staging()
    dE = torch.empty(n_sys, dtype=torch.float64, device="cuda")

    def one_pass():
        e.set_state(d_pos, d_vel, d_mass, stream=stream)
        e.integrate(ens.HERMITE, c.dt, c.steps, stream=stream)
        ens._check(ens.lib().ens_energy(e._h, dE.data_ptr(), None, ens.DEVICE, stream.cuda_stream), "ens_energy")

    with torch.cuda.stream(stream):
        for _ in range(args.warmup):
            one_pass()
        barrier()
        launches0 = e.info()["launches"]
        step_ms, kern_ms = [], []
        with ClockSampler(local) as clk:
            t_wall0 = time.perf_counter()
            for _ in range(args.steps):
                flush.zero_()  # L2 flush between timed iterations (outside the event pair)
                ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                ev0.record(stream)
                one_pass()
                ev1.record(stream)
                ev1.synchronize()
                step_ms.append(ev0.elapsed_time(ev1))
                kern_ms.append(e.last_kernel_ms())
            barrier()
            t_wall = time.perf_counter() - t_wall0
        launches = e.info()["launches"] - launches0
        clocks = clk.summary()
        total_ms = torch.tensor([sum(step_ms)], dtype=torch.float64, device="cuda")
        if world > 1:
            dist.all_reduce(total_ms, op=dist.ReduceOp.MAX)
        total_ms = float(total_ms.item())
        ms_per_step = total_ms / args.steps
        # work = the steps the systems actually took in a pass (a system a monitor stops early counts for what it ran)
        st = e.get_state(stream=stream)
        taken = torch.tensor([int(st["nsteps"].sum())], dtype=torch.float64, device="cuda")
        hist = np.bincount(st["status"], minlength=7).astype(np.int64)
        hist_t = torch.from_numpy(hist).cuda()
        if world > 1:
            dist.all_reduce(taken, op=dist.ReduceOp.SUM)
            dist.all_reduce(hist_t, op=dist.ReduceOp.SUM)
        taken_all, hist = float(taken.item()), hist_t.cpu().numpy()
        assert (st["nsteps"][st["status"] == ens.DONE_STEPS] == c.steps).all()
        if CFG == 1:  # the metric's ensemble fires no monitor: every system runs its full budget
            assert (st["status"] == ens.DONE_STEPS).all(), np.bincount(st["status"])
        value = taken_all / (ms_per_step * 1e-3)
        info = e.info()

        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic",
            "config": {"workload": c.name, "integrator": "hermite", "n_sys_per_gpu": n_sys, "n_body": n_body, "dt": c.dt,
                       "steps_per_launch": c.steps, "monitors": {"r_close": c.r_close, "r_eject": c.r_eject},
                       "l2": "flushed between timed iterations (512 MB memset); state lives in registers",
                       "parallelism": f"independent ensembles x{world}" if world > 1 else "single GPU"},
            "clocks": clocks, "gpu_launches": launches,
            "system_steps_per_pass": taken_all,
            "status_histogram": {name: int(hist[k]) for k, name in enumerate(
                ("active", "done_time", "done_steps", "stop_close", "stop_eject", "stop_nonfinite", "stop_stepsize")) if hist[k]},
            # context only (other hardware, derived): never the target, never vs_baseline
            "paper_context": {"m2070_system_steps_per_s_derived": 3.65e6, "source": "P:L347 Table 3 / P:L321"}, "wall_s_timed_region": t_wall,
            "pair_interactions_per_s": value * (n_body * (n_body - 1) // 2) * 3,
            "kernel": {"lanes_per_system": info["lanes_per_system"], "bodies_per_lane": info["bodies_per_lane"],
                       "threads": info["threads"], "blocks": info["blocks"], "regs": info["regs"],
                       "stack_bytes": info["stack_bytes"], "blocks_per_sm": info["blocks_per_sm"]},
        }

        peak_inst, peak_tf = nominal_fp64_peak(props.multi_processor_count, clocks.get("sm_max_mhz") or 1965.0)
        if rank == 0:
            instr, flops = hermite_work(n_body)
            k_ms = statistics.mean(kern_ms)
            per_rank = taken_all / world
            ach_tf = flops * per_rank / (k_ms * 1e-3) / 1e12
            prof = os.path.join("profiles", f"r2_hermite_cfg{CFG}_ncu_full.txt")
            roof = {"bound": "alu", "kernel": f"hermite_kernel<{n_body},{info['lanes_per_system']},{info['bodies_per_lane']}>"
                    + (" (time-sliced persistent grid)" if info["sliced"] else ""),
                    "achieved": ach_tf, "peak": peak_tf, "unit": "TFLOP/s", "frac": ach_tf / peak_tf,
                    # dram__bytes_read.sum + dram__bytes_write.sum of this kernel, one launch, read from the committed ncu
                    # summary of the same command (not measured in this run; null when that file is absent)
                    "traffic": profile_traffic(os.path.join(ROOT, prof)), "traffic_source": prof,
                    "algorithmic_hbm_bytes_per_launch": n_sys * ((13 * n_body + 2) * 8 + 12),
                    "peak_source": f"derived: {props.multi_processor_count} SMs x {FP64_LANES_PER_SM} FP64 lanes x 2 flop x "
                                   f"{clocks.get('sm_max_mhz') or 1965.0:.0f} MHz (DESIGN.md §8)",
                    "kernel_ms": k_ms, "algorithmic_fp64_instr_per_system_step": instr,
                    "algorithmic_flops_per_system_step": flops,
                    "achieved_lane_instr_per_s": instr * per_rank / (k_ms * 1e-3),
                    "issue_frac_nominal": instr * per_rank / (k_ms * 1e-3) / peak_inst}
            line["roofline"] = roof

        if not args.no_extras:
            # measured FP64 peak (DFMA chains), same box, same run
            peak_meas = ens.fp64_peak(100000, stream=stream)
            if rank == 0:
                line["roofline"]["peak_measured_lane_fma_per_s"] = peak_meas
                line["roofline"]["issue_frac_measured"] = line["roofline"]["achieved_lane_instr_per_s"] / peak_meas
            # e2e: host (pinned) buffers in, host buffers out, through the same C ABI calls
            out = {"pos": torch.empty_like(h_pos).pin_memory(), "vel": torch.empty_like(h_vel).pin_memory(),
                   "time": torch.empty(n_sys, dtype=torch.float64).pin_memory(),
                   "status": torch.empty(n_sys, dtype=torch.int32).pin_memory(),
                   "nsteps": torch.empty(n_sys, dtype=torch.int64).pin_memory()}
            hE = torch.empty(n_sys, dtype=torch.float64).pin_memory()

            def e2e_pass():
                e.set_state(h_pos, h_vel, h_mass, stream=stream)
                e.integrate(ens.HERMITE, c.dt, c.steps, stream=stream)
                e.get_state(stream=stream, out=out)
                ens._check(ens.lib().ens_energy(e._h, hE.data_ptr(), None, ens.HOST, stream.cuda_stream), "ens_energy")

            e2e_pass()
            barrier()
            n_e2e = max(3, min(args.steps, 5))
            t0 = time.perf_counter()
            for _ in range(n_e2e):
                e2e_pass()
            torch.cuda.synchronize()
            e2e_t = torch.tensor([time.perf_counter() - t0], dtype=torch.float64, device="cuda")
            if world > 1:
                dist.all_reduce(e2e_t, op=dist.ReduceOp.MAX)
            h2d = n_sys * n_body * 7 * 8
            d2h = n_sys * (n_body * 6 * 8 + 8 + 4 + 8 + 8)
            line["e2e"] = {"value": world * float(out["nsteps"].sum()) * n_e2e / float(e2e_t.item()), "unit": UNIT,
                           "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h, "passes": n_e2e,
                           "timing": "host wall clock around ens_set_state(HOST) + ens_integrate + ens_get_state(HOST) + "
                                     "ens_energy(HOST), pinned buffers"}

            def guarded(fn):
                try:
                    return fn()
                except ens.EnsError as ex:
                    return {"unavailable": str(ex)}

            # every other step-loop kernel, each with its own roofline figures
            others = {}
            for name, mk in others_table().items():
                if name == c.name:
                    continue
                kind, integ, arrays, nb, dt, steps, kw = mk()
                others[name] = guarded(lambda: time_kernel(ens, torch, stream, kind, integ, arrays, nb, dt, steps,
                                                           peak_inst, peak_tf, **kw))
                del arrays
            line["other_workloads"] = others
            if W.CONFIGS[4].name in others:
                line["mvs"] = dict(others[W.CONFIGS[4].name], workload=W.CONFIGS[4].name)

            # the paper's own workload shapes (section 5.1 initial conditions; Table 3: 131072 systems,
            # n = 3, 4, 5, 6, 10; fixed-step Hermite at the paper's dt = 1e-3).  Context beside it, never a target.
            shapes = {}
            for nb in (3, 4, 5, 6, 10):
                steps = max(100, int(2.3e6 / hermite_work(nb)[0]) // 100 * 100)  # ~20 ms kernels
                arrays = W.paper_ics(nb, n_sys=131072)
                shapes[f"hermite_paper_ics_131072x{nb}"] = guarded(lambda: time_kernel(
                    ens, torch, stream, "hermite", ens.HERMITE, arrays, nb, 1e-3, steps, peak_inst, peak_tf))
                del arrays
            line["paper_shapes"] = shapes

            # every dispatch shape of every fixed-step kernel (n_body = 2 .. 16): the tuning table of DESIGN.md section 8
            all_n = {}
            for nb in range(2, 17):
                ns = 131072 if nb <= 6 else 32768 if nb <= 10 else 8192
                arrays = W.paper_ics(nb, n_sys=ns)
                row = {"n_sys": ns}
                for kind, integ, dt in (("hermite", ens.HERMITE, 1e-3), ("hermite_carry", ens.HERMITE_CARRY, 1e-3),
                                        ("rkck", ens.RKCK, 1e-3), ("mvs", ens.MVS, 1e-2)):
                    steps = max(50, int(1.5e11 / (ns * WORK[kind](nb)[0])))  # ~10 ms kernels
                    r = guarded(lambda: time_kernel(ens, torch, stream, kind, integ, arrays, nb, dt, steps, peak_inst,
                                                    peak_tf, reps=2))
                    row[kind] = {k: r[k] for k in ("kernel_ms", "value", "issue_frac_nominal", "regs", "stack_bytes",
                                                   "lanes_per_system", "bodies_per_lane", "steps_taken") if k in r} or r
                all_n[str(nb)] = row
                del arrays
            line["all_n"] = all_n

            # HBM side of the path (rows a1 / a8 and the boundary kernels): achieved GB/s against MEASURED_PEAKS.json's
            # copy bandwidth, on the metric's ensemble and on one 16x larger (small launches are latency-bound)
            try:
                with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
                    hbm_peak = float(json.load(f)["hbm_gbs"])
            except Exception:
                hbm_peak = None
            hbm = {"peak_gbs": hbm_peak, "peak_source": "MEASURED_PEAKS.json hbm_gbs" if hbm_peak else "unavailable"}
            for tag, ns in ((f"{n_sys}x{n_body}", n_sys), (f"{16 * n_sys}x{n_body}", 16 * n_sys)):
                try:
                    pk, vk, mk = (torch.from_numpy(x).cuda() for x in W.generate(CFG, n_sys=ns, offset=lo))
                    ek = ens.Ensemble(ns, n_body)
                    outk = {"pos": torch.empty_like(pk), "vel": torch.empty_like(vk),
                            "time": torch.empty(ns, dtype=torch.float64, device="cuda"),
                            "status": torch.empty(ns, dtype=torch.int32, device="cuda"),
                            "nsteps": torch.empty(ns, dtype=torch.int64, device="cuda")}
                    Ek = torch.empty(ns, dtype=torch.float64, device="cuda")

                    def timed(fn, reps=5):
                        best = None
                        for _ in range(reps):
                            flush.zero_()
                            t0, t1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                            t0.record(stream)
                            fn()
                            t1.record(stream)
                            t1.synchronize()
                            best = t0.elapsed_time(t1) if best is None else min(best, t0.elapsed_time(t1))
                        return best * 1e-3

                    nb8 = n_body * 8
                    legs = {
                        # AoS read + SoA write of pos, vel, mass, plus the time/status/nsteps/nreject reset
                        "set_state": (lambda: ek.set_state(pk, vk, mk, stream=stream), ns * (2 * 7 * nb8 + 28)),
                        # zero steps: every row read once and written once by the step-loop kernel (a1 + a8)
                        "integrate_0_steps": (lambda: ek.integrate(ens.HERMITE, c.dt, 0, stream=stream),
                                              ns * ((13 * n_body + 2) * 8 + 12)),
                        "get_state": (lambda: ek.get_state(stream=stream, out=outk), ns * (2 * 6 * nb8 + 2 * 20)),
                        "energy": (lambda: ens._check(ens.lib().ens_energy(ek._h, Ek.data_ptr(), None, ens.DEVICE,
                                                                          stream.cuda_stream), "ens_energy"),
                                   ns * (7 * nb8 + 8)),
                    }
                    ek.set_state(pk, vk, mk, stream=stream)
                    hbm[tag] = {}
                    for name, (fn, nbytes) in legs.items():
                        sec = timed(fn)
                        hbm[tag][name] = {"us": sec * 1e6, "gbs": nbytes / sec / 1e9,
                                          "frac": (nbytes / sec / 1e9 / hbm_peak) if hbm_peak else None}
                    ek.close()
                    del pk, vk, mk, outk, Ek
                except ens.EnsError as ex:
                    hbm[tag] = {"unavailable": str(ex)}
            line["hbm"] = hbm

    if rank == 0 and not args.no_cpu_baseline and world == 1:
        line["cpu_baseline"] = cpu_baseline()
    if rank == 0:
        print(json.dumps(line), flush=True)
    e.close()
    if world > 1:
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
