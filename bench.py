#!/usr/bin/env python
"""bench.py — BASELINE.json's metric on BASELINE.json's headline config, through the C ABI of libens.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]

Metric: Hermite FP64 system-steps/s on config 1 (131072 systems x 3 bodies, dt = 0.01, 10^4 steps per launch, close
approach and ejection monitors armed).  One bench "step" is one pass of the hot path over the whole ensemble:
ens_set_state (AoS -> SoA, inputs already resident in HBM) -> ens_integrate(HERMITE, 10^4 steps: load, 3 x
acc+jerk, predictor, 2 x corrector, monitors, retire, store) -> ens_energy.  `value` = n_sys * 10^4 * n_gpus /
seconds per step.  `e2e` is the same pass through HOST buffers (pinned), host<->device copies inside the timed region.
The MVS kernel (config 4) and the roofline of the dominant kernel are reported in the same JSON line.

N > 1 (torchrun): every rank integrates its own config-1 ensemble (different system indices, no data-path
collective: systems are independent) -> weak scaling; time = max over ranks.
`--impl reference` times the CPU oracle (rank 0 only) on a bounded sample of the same workload.
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

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from paper_1208_1157_b200 import workloads as W  # noqa: E402

METRIC = "hermite_fp64_system_steps_per_sec_131072x3"
UNIT = "system-steps/s"
CFG = 1

# Algorithmic FP64 work of one Hermite system-step: each unordered pair once per evaluation,
# 3 evaluations per step; FMA = 2 flops, add/mul = 1.
PAIR_INSTR, PAIR_FLOPS = 38, 60           # one pair acc+jerk evaluation
COMP_INSTR, COMP_FLOPS = 17, 34           # predictor + 2 correctors, per body component
BODY_MON_INSTR, BODY_MON_FLOPS = 3, 5     # |x_i|^2 for the ejection monitor


def hermite_work(n_body: int):
    pairs = n_body * (n_body - 1) // 2
    instr = 3 * pairs * PAIR_INSTR + 3 * n_body * COMP_INSTR + n_body * BODY_MON_INSTR + 1
    flops = 3 * pairs * PAIR_FLOPS + 3 * n_body * COMP_FLOPS + n_body * BODY_MON_FLOPS + 1
    return instr, flops


# FP64 peak of a B200: 148 SMs x 64 FP64 lanes x 1 FMA/clk x max SM clock.
FP64_LANES_PER_SM = 64


def nominal_fp64_peak(sm_count: int, sm_max_mhz: float):
    lane_inst = sm_count * FP64_LANES_PER_SM * sm_max_mhz * 1e6
    return lane_inst, 2.0 * lane_inst / 1e12  # lane-instr/s, TFLOP/s


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


def cpu_baseline(budget_s: float = 12.0):
    """The oracle, as it stands, on this box's host cores, on a bounded sample of config 1 (full 10^4 steps each)."""
    import oracle
    c = W.CONFIGS[CFG]
    cores = oracle.host_cores()
    pos, vel, mass = W.generate(CFG, n_sys=16 * cores)
    t0 = time.perf_counter()
    oracle.integrate(oracle.HERMITE, pos, vel, mass, dt=c.dt, max_steps=1000, r_close=c.r_close, r_eject=c.r_eject,
                     nthreads=cores)
    rate = 16 * cores * 1000 / (time.perf_counter() - t0)  # calibration only
    n = int(max(cores, min(c.n_sys, rate * budget_s / c.steps)))
    n = max(cores, n // cores * cores)
    pos, vel, mass = W.generate(CFG, n_sys=n)
    t0 = time.perf_counter()
    oracle.integrate(oracle.HERMITE, pos, vel, mass, dt=c.dt, max_steps=c.steps, r_close=c.r_close,
                     r_eject=c.r_eject, nthreads=cores)
    dt = time.perf_counter() - t0
    return {"value": n * c.steps / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": f"first {n} systems of config 1 x {c.steps} steps ({dt:.1f} s wall, system-per-thread OpenMP)"}, dt


def run_reference(args):
    """--impl reference: the CPU oracle (rank 0 only), each step a bounded sample of config 1."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    import oracle
    c = W.CONFIGS[CFG]
    cores = oracle.host_cores()
    n = 32 * cores
    pos, vel, mass = W.generate(CFG, n_sys=n)
    sub = 2000  # steps per sample: 32 systems per core x 2000 steps ~ 0.1 s per bench step per core-GHz
    run = lambda: oracle.integrate(oracle.HERMITE, pos, vel, mass, dt=c.dt, max_steps=sub, r_close=c.r_close,
                                   r_eject=c.r_eject, nthreads=cores)
    for _ in range(args.warmup):
        run()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        run()
    dt = time.perf_counter() - t0
    value = n * sub * args.steps / dt
    sample = f"{n} systems of config 1 x {sub} steps per bench step"
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": dt / args.steps * 1e3, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": W.CONFIGS[CFG].name, "integrator": "hermite", "dt": c.dt, "sample": sample},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=1, choices=[0, 1, 2, 3],
                    help="Hermite workload (BASELINE.json configs index); 1 is the metric's, the others are for profiling")
    ap.add_argument("--no-cpu-baseline", action="store_true", help="skip the oracle timing leg (profiling runs)")
    ap.add_argument("--no-extras", action="store_true", help="skip the MVS / e2e / peak legs (profiling runs)")
    args = ap.parse_args()
    global CFG, METRIC
    if args.config != CFG:
        CFG = args.config
        METRIC = "hermite_fp64_system_steps_per_sec_" + W.CONFIGS[CFG].name.split("_", 1)[1]
    if args.impl == "reference":
        return run_reference(args)
    args.warmup = max(args.warmup, 3)

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

    c = W.CONFIGS[CFG]
    n_sys, n_body = c.n_sys, c.n_body
    # each rank owns its own range of system indices of the same seeded generator (weak scaling, no exchange)
    from paper_1208_1157_b200 import shard
    lo, hi = shard.weak_range(n_sys, rank)
    pos, vel, mass = W.generate(CFG, n_sys=hi - lo, offset=lo)
    d_pos, d_vel, d_mass = (torch.from_numpy(x).cuda() for x in (pos, vel, mass))
    h_pos, h_vel, h_mass = (torch.from_numpy(x).pin_memory() for x in (pos, vel, mass))
    stream = torch.cuda.Stream()
    flush = torch.empty(512 * 1024 * 1024 // 4, dtype=torch.int32, device="cuda")  # 512 MB > 126 MB L2
    e = ens.Ensemble(n_sys, n_body)
    e.set_monitors(c.r_close, c.r_eject)
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
        value = world * n_sys * c.steps / (ms_per_step * 1e-3)
        st = e.get_state(stream=stream)
        assert (st["nsteps"][st["status"] == ens.DONE_STEPS] == c.steps).all()
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
            # context only (other hardware, derived): never the target, never vs_baseline
            "paper_context": {"m2070_system_steps_per_s_derived": 3.65e6, "source": "P:L347 Table 3 / P:L321"}, "wall_s_timed_region": t_wall,
            "pair_interactions_per_s": value * (n_body * (n_body - 1) // 2) * 3,
            "kernel": {"lanes_per_system": info["lanes_per_system"], "bodies_per_lane": info["bodies_per_lane"],
                       "threads": info["threads"], "blocks": info["blocks"], "regs": info["regs"],
                       "blocks_per_sm": info["blocks_per_sm"]},
        }

        if rank == 0:
            props = torch.cuda.get_device_properties(local)
            instr, flops = hermite_work(n_body)
            k_ms = statistics.mean(kern_ms)
            peak_inst, peak_tf = nominal_fp64_peak(props.multi_processor_count, clocks.get("sm_max_mhz") or 1965.0)
            ach_tf = flops * n_sys * c.steps / (k_ms * 1e-3) / 1e12
            roof = {"bound": "alu", "kernel": f"hermite_kernel<{n_body},{info['lanes_per_system']},{info['bodies_per_lane']}>", "achieved": ach_tf, "peak": peak_tf, "unit": "TFLOP/s",
                    "frac": ach_tf / peak_tf,
                    # ncu dram__bytes_read.sum + dram__bytes_write.sum of this kernel, one launch, config 1
                    # (profiles/r1i_hermite_cfg1_ncu_full.txt); the store drains from L2 after the kernel ends
                    "traffic": 24.7e6 if CFG == 1 else None,
                    "peak_source": f"derived: {props.multi_processor_count} SMs x {FP64_LANES_PER_SM} FP64 lanes x 2 flop x "
                                   f"{clocks.get('sm_max_mhz') or 1965.0:.0f} MHz (DESIGN.md §8)",
                    "kernel_ms": k_ms, "algorithmic_fp64_instr_per_system_step": instr,
                    "algorithmic_flops_per_system_step": flops,
                    "achieved_lane_instr_per_s": instr * n_sys * c.steps / (k_ms * 1e-3),
                    "issue_frac_nominal": instr * n_sys * c.steps / (k_ms * 1e-3) / peak_inst}
            line["roofline"] = roof

        if not args.no_extras:
            # measured FP64 peak (DFMA chains), same box, same run
            peak_meas = ens.fp64_peak(100000, stream=stream)
            if rank == 0:
                line["roofline"]["peak_measured_lane_fma_per_s"] = peak_meas
                line["roofline"]["issue_frac_measured"] = line["roofline"]["achieved_lane_instr_per_s"] / peak_meas
            # e2e: host (pinned) buffers in, host buffers out, through the same C ABI calls
            out = {"pos": torch.empty_like(h_pos), "vel": torch.empty_like(h_vel),
                   "time": torch.empty(n_sys, dtype=torch.float64).pin_memory(),
                   "status": torch.empty(n_sys, dtype=torch.int32).pin_memory(),
                   "nsteps": torch.empty(n_sys, dtype=torch.int64).pin_memory()}
            out["pos"], out["vel"] = out["pos"].pin_memory(), out["vel"].pin_memory()
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
            line["e2e"] = {"value": world * n_sys * c.steps * n_e2e / float(e2e_t.item()), "unit": UNIT,
                           "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h, "passes": n_e2e,
                           "timing": "host wall clock around ens_set_state(HOST) + ens_integrate + ens_get_state(HOST) + "
                                     "ens_energy(HOST), pinned buffers"}
            # the other kernels of the path, each on its own BASELINE.json config at full size (kernel time only; not
            # part of the metric): Hermite n_body = 6 and 15, and the second kernel, MVS on config 4
            others = {}
            for k in (2, 3, 4):
                if k == CFG:
                    continue
                ck = W.CONFIGS[k]
                try:
                    pk, vk, mk = (torch.from_numpy(x).cuda() for x in W.generate(k, offset=rank * ck.n_sys))
                    ek = ens.Ensemble(ck.n_sys, ck.n_body)
                    ek.set_monitors(ck.r_close, ck.r_eject)
                    msk = []
                    for _ in range(3):
                        ek.set_state(pk, vk, mk, stream=stream)
                        ek.integrate(ck.integrator, ck.dt, ck.steps, stream=stream)
                        msk.append(ek.last_kernel_ms())
                    ik, tk = ek.info(), min(msk[1:])
                    o = {"value": ck.n_sys * ck.steps / (tk * 1e-3), "unit": "system-steps/s", "kernel_ms": tk,
                         "regs": ik["regs"], "lanes_per_system": ik["lanes_per_system"],
                         "bodies_per_lane": ik["bodies_per_lane"], "blocks_per_sm": ik["blocks_per_sm"]}
                    if ck.integrator == W.HERMITE:
                        ins, _ = hermite_work(ck.n_body)
                        o["issue_frac_nominal"] = o["value"] * ins / nominal_fp64_peak(
                            torch.cuda.get_device_properties(local).multi_processor_count,
                            clocks.get("sm_max_mhz") or 1965.0)[0]
                    others[ck.name] = o
                    ek.close()
                    del pk, vk, mk
                except ens.EnsError as ex:
                    others[ck.name] = {"unavailable": str(ex)}
            # HBM side of the path (rows a1 / a8 and the boundary kernels): achieved GB/s against MEASURED_PEAKS.json's
            # copy bandwidth, on the metric's ensemble and on one 16x larger (small launches are latency-bound)
            try:
                with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
                    hbm_peak = float(json.load(f)["hbm_gbs"])
            except Exception:
                hbm_peak = None
            hbm = {"peak_gbs": hbm_peak, "peak_source": "MEASURED_PEAKS.json hbm_gbs" if hbm_peak else "unavailable"}
            for tag, ns in (("131072x3", n_sys), ("2097152x3", 16 * n_sys)):
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
                        # AoS read + SoA write of pos, vel, mass, plus the time/status/nsteps reset
                        "set_state": (lambda: ek.set_state(pk, vk, mk, stream=stream), ns * (2 * 7 * nb8 + 20)),
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
            # adaptive-step Hermite (Eq. 5) on the metric's own systems, tau = 0.017 to t = 20; event-timed
            # around the C-ABI call (ordering pre-pass + kernel); system-steps = steps actually taken
            try:
                ea = ens.Ensemble(n_sys, n_body)
                ea.set_monitors(c.r_close, c.r_eject)
                best = None
                for _ in range(3):
                    ea.set_state(d_pos, d_vel, d_mass, stream=stream)
                    a0, a1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                    a0.record(stream)
                    ea.integrate(ens.HERMITE_ADAPTIVE, 0.017, 10**9, t_end=20.0, stream=stream)
                    a1.record(stream)
                    a1.synchronize()
                    best = a0.elapsed_time(a1) if best is None else min(best, a0.elapsed_time(a1))
                taken = int(ea.get_state(stream=stream)["nsteps"].sum())
                others["hermite_adaptive_131072x3"] = {"value": taken / (best * 1e-3), "unit": "system-steps/s", "ms": best,
                                                       "tau": 0.017, "t_end": 20.0, "steps_taken": taken,
                                                       "regs": ea.info()["regs"]}
                ea.close()
            except ens.EnsError as ex:
                others["hermite_adaptive_131072x3"] = {"unavailable": str(ex)}
            # the 2-evaluation Hermite and the Cash-Karp kernels on the metric's own ensemble (kernel time, full 10^4 steps)
            for integ, key in ((ens.HERMITE_CARRY, "hermite_carry_131072x3"), (ens.RKCK, "rkck_131072x3")):
                try:
                    msk = []
                    for _ in range(2):
                        e.set_state(d_pos, d_vel, d_mass, stream=stream)
                        e.integrate(integ, c.dt, c.steps, stream=stream)
                        msk.append(e.last_kernel_ms())
                    others[key] = {"value": n_sys * c.steps / (msk[-1] * 1e-3), "unit": "system-steps/s",
                                   "kernel_ms": msk[-1], "regs": e.info()["regs"]}
                except ens.EnsError as ex:
                    others[key] = {"unavailable": str(ex)}
            line["other_workloads"] = others
            if W.CONFIGS[4].name in others:
                line["mvs"] = dict(others[W.CONFIGS[4].name], workload=W.CONFIGS[4].name)

    if rank == 0 and not args.no_cpu_baseline and world == 1:
        cb, _ = cpu_baseline()
        line["cpu_baseline"] = cb
    if rank == 0:
        print(json.dumps(line), flush=True)
    e.close()
    if world > 1:
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
