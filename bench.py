#!/usr/bin/env python
"""bench.py -- cell-updates/s of the 14-moment 2-D time step on the crossed-jet workload.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference] [--n 2048] [--kn 0.1]

A "step" is one pass of the whole hot path (ghost cells, cons->prim, MUSCL, closure fluxes +
wave speeds, HLL, update + BGK source, CFL reduction -> next dt) over BASELINE.json configs[3]:
2048 x 2048 cells, crossed Mach-3 jets, Kn = 0.1, seeded +-1% density perturbation, CFL 0.4.
Prints ONE JSON line (rank 0).  See DESIGN.md section 9 for how each field is obtained.

N > 1 (torchrun): the path has no multi-GPU exchange yet ("replicas only"):
every rank steps its own replica, value = all ranks' cell updates / max-over-ranks time.
`--impl reference` times the CPU oracle (test infrastructure) on a bounded sample instead.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parent
sys.path.insert(0, str(ROOT))

import mm_workloads as wl  # noqa: E402

METRIC = "cell-updates/s (fp64, 14-moment 2-D)"
UNIT = "cell-updates/s"
CFL = 0.4


def flops_per_cell_update(shared_limiter: bool, zsym: bool, system: int = 14, limiter: int = 1, flux: int = 0):
    """Algorithmic FP64 operations per cell update (each + - * / sqrt exp
    pow = 1, so a(P*), b(P*) of Eq 29c-d are 10 per call whatever the kernel's table evaluation executes).
    -> (count of the formulation the CUDA path runs, the same with the table evaluation as executed,
        count of the oracle's naive restatement).
    The roofline line uses the FIRST (smallest) number: flops the kernel does not execute, or executes
    only because of an implementation choice, are not credited to it.  All are produced by committed
    counting builds, not typed in."""
    from paper_2401_15233_b200 import build_ext
    # counted for the limiter and the flux function that ran (van Albada / Rusanov carry a key suffix, opcount.txt)
    key = (f"kernel_flops_per_cell_update_{system}_" + ("zsym_" if zsym and system == 14 else "")
           + ("shared_limiter" if shared_limiter else "per_variable_limiter")
           + ("_vanalbada" if limiter == wl.LIM_VANALBADA else "") + ("_rusanov" if flux == wl.FLUX_RUSANOV else ""))
    oc = build_ext.read_opcount()
    k = oc[key]
    o = None
    for line in (ROOT / "tests" / "golden" / "oracle_opcount.txt").read_text().splitlines():
        if line.startswith(f"flops_per_cell_update_{system} "):
            o = float(line.split()[1])
    return float(k), float(oc.get(key + "_executed", k)), o


# dram__bytes_read.sum + dram__bytes_write.sum of ONE launch of the dominant kernel, from the
# `ncu --set full` capture summarised in profiles/ (None where no capture of that configuration exists).
NCU_TRAFFIC_BYTES = {
    ("k_step14_tm<zsym>", 2048): (703.22e6 + 627.64e6, "profiles/r3_k_step14_tm_zsym.md"),
    ("k_step14_tm<general>", 2048): (975.68e6 + 898.51e6, "profiles/r3_k_step14_tm_general.md"),
}
FP64_LANES_PER_SM = 64      # DFMA lanes of a B200 SM: nominal peak = SMs x 64 x 2 flop x SM clock


def peaks() -> dict:
    f = ROOT / "MEASURED_PEAKS.json"
    return json.loads(f.read_text()) if f.exists() else {}


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 50 ms while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.rows, self.proc = index, [], None

    def __enter__(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "50",
                 "-i", str(self.index)], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except OSError:
            self.proc = None
        return self

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def __exit__(self, *a):
        if self.proc:
            time.sleep(0.25)
            self.proc.terminate()
            self.th.join(timeout=2)

    def summary(self) -> dict:
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1]))
            except (ValueError, IndexError):
                continue
            for k, nm in enumerate(names):
                if len(r) > 3 + k and r[3 + k].lower().startswith("active"):
                    reasons.add(nm)
        busy = [c for c in sm if c > 0.5 * max(sm)] if sm else []
        return {"sm_mhz": float(np.median(busy)) if busy else None,
                "sm_max_mhz": max(mx) if mx else None, "reasons": sorted(reasons),
                "samples": len(sm)}


def max_over_ranks(x: float, device) -> float:
    """Device-timed milliseconds -> max over all ranks (replicas finish when the slowest does)."""
    import torch
    import torch.distributed as dist
    if not dist.is_available() or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(x)
    t = torch.tensor([x], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def job_throughput(world: int, cells: int, steps: int, ms: float) -> float:
    """Whole-job cell-updates/s: every rank steps its own replica of `cells` cells."""
    return world * cells * steps / (ms * 1e-3)


WORKLOADS = {
    # name: (builder(n, kn), CFL, description)
    "baseline": (lambda n, kn: wl.crossed_jets(n, Kn=kn, perturb=0.01), 0.4,
                 "crossed jets {n}x{n}, 14-moment, Kn={kn}, +-1% seeded density perturbation, minmod (shared psi) "
                 "+ HLL, CFL 0.4 (BASELINE configs[3])"),
    "paper-crossing": (lambda n, kn: wl.paper_jets(n, two=True), 0.5,
                       "the paper's collisionless M=5 crossing jets {n}x{n} (PAPER.md L446-470), van Albada "
                       "(shared psi) + Rusanov, CFL 0.5; SURVEY 8(f) item 1, not the BASELINE metric's workload"),
    "paper-single": (lambda n, kn: wl.paper_jets(n, two=False), 0.5,
                     "the paper's collisionless M=5 single jet {n}x{n} (PAPER.md L430-444), van Albada (shared "
                     "psi) + Rusanov, CFL 0.5; SURVEY 8(f) item 1, not the BASELINE metric's workload"),
    "sod5": (lambda n, kn: wl.sod5(n, Kn=kn), 0.5,
             "1-D 5-moment Sod tube, {n} cells, Kn={kn}, minmod + HLL, CFL 0.5 (BASELINE configs[0] at n=1000, "
             "kn=0.01): a correctness config, far too small to load a GPU (launch-latency bound)"),
    "sod14": (lambda n, kn: wl.sod14(n, 4, Kn=kn), 0.5,
              "14-moment Sod tube on {n}x4 cells, periodic y, Kn={kn}, minmod + HLL, CFL 0.5 (BASELINE configs[1] "
              "at n=4096): a correctness config, 16 K cells"),
}
WORKLOAD = "baseline"


def workload(n: int, kn: float) -> dict:
    return WORKLOADS[WORKLOAD][0](n, kn)


def time_oracle(n: int, kn: float, steps: int, warmup: int = 0, nthreads: int = 0, ny: int = 0):
    """Oracle (as it stands) on an n x n instance of the workload: cell-updates/s, threads."""
    from oracle import mmo
    prob = workload(n, kn)
    if ny and ny < prob["ny"]:          # a band of rows around the lower jet (same cells, same boundary data)
        j0 = max(0, min(prob["ny"] - ny, int(0.35 * prob["ny"]) - ny // 2))
        y0, y1 = prob["extent"][2], prob["extent"][3]
        h = (y1 - y0) / prob["ny"]
        prob = dict(prob, ny=ny, W0=np.ascontiguousarray(prob["W0"][:, j0:j0 + ny]),
                    extent=(prob["extent"][0], prob["extent"][1], y0 + j0 * h, y0 + (j0 + ny) * h))
    so = mmo.Solver(prob["system"], prob["nx"], prob["ny"], extent=prob["extent"],
                    collision=prob["collision"], bcs=prob["bcs"], nthreads=nthreads, **prob["options"])
    so.set_state_prim(prob["W0"])
    if warmup:
        so.step(warmup, CFL)
    t0 = time.perf_counter()
    so.step(steps, CFL)
    dt = time.perf_counter() - t0
    return prob["nx"] * prob["ny"] * steps / dt, so.threads, dt


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    n = args.ref_n
    val, threads, secs = time_oracle(n, args.kn, args.steps, args.warmup)
    sample = f"{n}x{n} instance of the crossed-jet workload, {args.steps} CFL steps ({secs:.1f} s)"
    out = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
           "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * secs / max(args.steps, 1),
           "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
           "data": "synthetic", "gpu_launches": 0,
           "config": {"workload": WORKLOADS[WORKLOAD][2].format(n=args.n, kn=args.kn)
                                  + f"; oracle timed on a bounded {n}x{n} sample of it"},
           "cpu_baseline": {"value": val, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample},
           "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(out), flush=True)


def run_gpu_batch5(args):
    """--workload sod5-batch: `--tubes` independent 5-moment Sod tubes of `--n` cells, sigma_lim x Kn
    sweep values cycled over the tubes (section 4.3).  Single GPU."""
    import torch
    from paper_2401_15233_b200 import mm
    torch.cuda.set_device(0)
    nx, nt, K, W = args.n, args.tubes, args.steps, args.warmup
    sig = np.resize([1e-2, 1e-3, 1e-4, 1e-5], nt)
    kns = np.resize(np.repeat([1e-3, 1e-2, 1e-1, 1.0, 0.0], 4), nt)
    W0 = wl.sod5(nx, Kn=0.01)["W0"].reshape(5, nx)
    b = mm.Batch5(nx, sig, kns)
    cells = nx * nt
    b.set_state_prim(W0)
    b.step(W, 0.5)
    torch.cuda.synchronize()
    l0 = b.launches
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    with ClockSampler(0) as clk:
        ev0.record(); b.step(K, 0.5); ev1.record()
        torch.cuda.synchronize()
    ms = ev0.elapsed_time(ev1)
    launches = b.launches - l0
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(); b.set_state_prim(W0); b.step(K, 0.5); U = b.get_state(); e1.record()
    torch.cuda.synchronize()
    e2e_ms = e0.elapsed_time(e1)
    from paper_2401_15233_b200 import build_ext
    fpc = float(build_ext.read_opcount()["kernel_flops_per_cell_update_5_per_variable_limiter"])
    peak_tf = mm.mm_measure_fp64_peak(5)
    achieved = fpc * cells * K / (ms * 1e-3) * 1e-12          # finalize kernel (ntubes threads) included
    inf = b.info(check=False)
    print(json.dumps({
        "metric": "cell-updates/s (fp64, 5-moment 1-D, batched tubes)", "value": cells * K / (ms * 1e-3),
        "unit": UNIT, "n_gpus": 1, "steps": K, "warmup": W, "ms_per_step": ms / K, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": f"{nt} independent 5-moment Sod tubes x {nx} cells, sigma_lim in 1e-2..1e-5, Kn in "
                               f"1e-3..1 and collisionless, minmod + HLL, own CFL 0.5 time step per tube "
                               f"(SURVEY 8(f) item 4; not the BASELINE metric's workload)",
                   "cells": cells, "state_finite": bool(np.isfinite(U).all()), "tubes_failed": int(inf["failed"].sum())},
        "clocks": clk.summary(),
        "e2e": {"value": cells * K / (e2e_ms * 1e-3), "unit": UNIT, "h2d_bytes_per_step": W0.nbytes / K,
                "d2h_bytes_per_step": U.nbytes / K},
        "gpu_launches": launches,
        "roofline": {"bound": "alu", "achieved": achieved, "peak": peak_tf, "unit": "TFLOP/s",
                     "frac": achieved / peak_tf, "traffic": None, "kernel": "k_batch5_step",
                     "flops_per_cell_update": fpc},
        "cpu_baseline": None}), flush=True)


def run_gpu(args):
    import torch
    import torch.distributed as dist
    from paper_2401_15233_b200 import mm

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the library has no CPU path)")
    torch.cuda.set_device(local)
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    n, K, W = args.n, args.steps, args.warmup
    prob = workload(n, args.kn)
    nm = prob["system"]
    cells = prob["nx"] * prob["ny"]
    s = mm.Solver.from_problem(prob, load_state=False, device=f"cuda:{local}")
    nbytes_state = nm * cells * 8
    W_host = torch.from_numpy(prob["W0"]).pin_memory()
    U_host = torch.empty((nm, prob["ny"], prob["nx"]), dtype=torch.float64).pin_memory()
    W_dev = W_host.to(f"cuda:{local}")

    if args.general_path:
        s.set_fast_path(False)
    # ---- device-resident timing: K steps, inputs in HBM (two 470 MB copies >> 126 MB L2)
    s.set_state_prim(W_dev)
    developed = None
    if args.developed_t > 0.0:          # timed window on a developed state: CFL steps to t first
        s.advance_to(args.developed_t, CFL)
        developed = s.info(check=False)
    s.step(W, CFL)
    barrier()
    l0 = s.launches
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    with ClockSampler(local) as clk:
        ev0.record(s.stream)
        s.step(K, CFL)
        ev1.record(s.stream)
        barrier()
    ms = ev0.elapsed_time(ev1)
    launches = s.launches - l0
    # the dominant kernel's own duration: a second, shorter run of the same steps with CUDA events
    # around every step-kernel launch (kept out of the timed region: the event records sit between
    # the two kernels of a step and would serialise their launch overlap)
    s.profile_begin()
    s.step(min(K, 200), CFL)
    barrier()
    kern_ms, kern_n = s.profile_end()
    info = s.info()
    ms = max_over_ranks(ms, f"cuda:{local}")
    value = job_throughput(world, cells, K, ms)

    # ---- end to end through the API with HOST buffers: H2D of the state, K steps, D2H of the result
    barrier()
    t0 = time.perf_counter()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(s.stream)
    s.set_state_prim(W_host)
    s.step(K, CFL)
    s.get_state(U_host)
    e1.record(s.stream)
    barrier()
    e2e_ms = e0.elapsed_time(e1)
    e2e_ms = max_over_ranks(e2e_ms, f"cuda:{local}")
    e2e_value = job_throughput(world, cells, K, e2e_ms)
    finite = bool(torch.isfinite(U_host).all())

    if rank == 0:
        opt = prob["options"]
        fpc, fpc_exec, fpc_oracle = flops_per_cell_update(bool(opt["shared_limiter"]), s.fast_path_active, nm,
                                                          limiter=opt["limiter"], flux=opt["flux"])
        # the probe also reports the SM clock it ran at (cycle counter / global timer inside the kernel)
        peak_tf, peak_mhz = mm.mm_measure_fp64_peak(5, with_clock=True)
        # the pipe's instruction rates when the register-reuse cache cannot supply operands
        r_dfma3, r_dmul, r_dadd = mm.mm_measure_fp64_operand_rates(3)
        sms = torch.cuda.get_device_properties(local).multi_processor_count
        nominal_tf = sms * FP64_LANES_PER_SM * 2.0 * (peak_mhz or 0.0) * 1e6 * 1e-12
        kern_avg_ms = kern_ms / max(kern_n, 1)
        achieved_tf = fpc * cells / (kern_avg_ms * 1e-3) * 1e-12
        pk = peaks()
        hbm_gbs = 16.0 * nm * cells / (kern_avg_ms * 1e-3) * 1e-9
        # what the kernel really moves: U and W(U) are both resident, i.e. read NV + NV and
        # write NV + NV doubles per cell update with NV = 10 carried moments on the z-symmetric variant, 14 on the
        # general one; the 5-moment kernel reads 5 and writes 5
        nv = 5 if nm == 5 else (10 if s.fast_path_active else 14)
        moved_model = 8.0 * (2 * nv if nm == 5 else 4 * nv) * cells
        cpu = None
        if world == 1 and not args.no_cpu_baseline:
            v, threads, secs = time_oracle(args.ref_n, args.kn, args.cpu_steps)
            # the paper's own baseline is ONE core: the same oracle, one thread, on a
            # 128-row band of the same instance
            v1, t1, s1 = time_oracle(args.ref_n, args.kn, args.cpu_steps_single, nthreads=1, ny=128)
            cpu = {"value": v, "unit": UNIT, "cores": threads, "kind": "oracle",
                   "sample": f"{args.ref_n}x{args.ref_n} instance of the same workload, "
                             f"{args.cpu_steps} CFL steps ({secs:.1f} s)",
                   "single_thread": {"value": v1, "unit": UNIT, "cores": t1,
                                     "sample": f"{args.ref_n}x128 band of that instance around the lower jet, "
                                               f"{args.cpu_steps_single} CFL steps ({s1:.1f} s)"}}
        kernel_name = ("k_step5" if nm == 5 else
                       "k_step14_tm<zsym>" if s.fast_path_active else "k_step14_tm<general>")
        traffic, traffic_src = NCU_TRAFFIC_BYTES.get((kernel_name, n), (None, None)) if WORKLOAD == "baseline" else (None, None)
        out = {
            "metric": METRIC if nm == 14 else "cell-updates/s (fp64, 5-moment 1-D)",
            "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
            "ms_per_step": ms / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": {"workload": WORKLOADS[WORKLOAD][2].format(n=n, kn=args.kn),
                       "cells": cells, "l2": (f"inputs larger than L2 (2 x {nbytes_state / 1e6:.0f} MB state copies)" if nbytes_state > 126e6
                              else f"L2-resident state ({nbytes_state / 1e6:.2f} MB): not a bandwidth measurement"),
                       "parallelism": "replicas only" if world > 1 else "single GPU",
                       "t_end": info["t"], "state_finite": finite,
                       "window": (f"developed state: {developed['steps']} CFL steps to t = {developed['t']:.4g} before "
                                  f"the warm-up (status {developed['status']})" if developed else
                                  "starting state of the config + warm-up steps")},
            "clocks": clk.summary(),
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": nbytes_state / K,
                    "d2h_bytes_per_step": nbytes_state / K,
                    "note": f"one job = H2D of the {nbytes_state} B state from pinned memory + {K} steps + "
                            f"D2H of the result; bytes amortised over the {K} steps"},
            "gpu_launches": launches,
            "roofline": {"bound": "alu", "achieved": achieved_tf, "peak": peak_tf, "unit": "TFLOP/s",
                         "frac": achieved_tf / peak_tf if peak_tf else None,
                         "traffic": traffic, "traffic_unit": "bytes per launch (ncu dram read + write)",
                         "traffic_source": traffic_src, "algorithmic_bytes_per_launch": 16.0 * nm * cells,
                         "algorithmic_bytes_note": "SURVEY 8(d): read 14 + write 14 doubles per cell update; the 14-moment kernel "
                                                   "keeps U and W(U) resident and moves 2 x (10 + 10) doubles on the z-symmetric "
                                                   "variant (2 x 28 on the general one), DESIGN.md section 6",
                         "kernel": kernel_name,
                         "kernel_ms": kern_avg_ms,
                         "flops_per_cell_update": fpc, "flops_per_cell_update_executed": fpc_exec,
                         "flops_per_cell_update_oracle": fpc_oracle,
                         "flops_convention": "SURVEY.md 8(d): + - * / sqrt exp pow = 1 each, FMA = 2; a(P*), b(P*) of "
                                             "Eq 29c-d booked as the method's formulas, not as the table evaluation",
                         "peak_source": "best of two register-resident FP64 DFMA loops measured in this run (multiplier in a "
                                        "register / as an instruction immediate; mm_measure_fp64_peak, libmm_bench.so)",
                         "peak_sm_mhz": peak_mhz, "peak_nominal": nominal_tf,
                         "fp64_operand_rates": {"unit": "1e12 thread instructions/s, operands from distinct registers",
                                                "dfma_three_registers": r_dfma3, "dmul": r_dmul, "dadd": r_dadd,
                                                "note": "a DFMA reading three distinct registers holds the pipe 3 cycles, "
                                                        "DMUL / DADD / DFMA with a reused or constant operand 2 "
                                                        "(mm_measure_fp64_operand_rates; DESIGN.md 9.3)"},
                         "frac_of_nominal": achieved_tf / nominal_tf if nominal_tf else None,
                         "hbm_algorithmic_gbs": hbm_gbs, "hbm_peak_gbs": pk.get("hbm_gbs"),
                         "hbm_algorithmic_frac": hbm_gbs / pk["hbm_gbs"] if pk.get("hbm_gbs") else None,
                         # bytes really moved per launch: the ncu capture where one exists, else the kernel's own count
                         "hbm_moved_bytes_per_launch": traffic if traffic else moved_model,
                         "hbm_moved_source": traffic_src if traffic else "2 x (NV + NV) doubles per cell update (U and W(U) resident)",
                         "hbm_moved_gbs": (traffic if traffic else moved_model) / (kern_avg_ms * 1e-3) * 1e-9,
                         "hbm_frac": ((traffic if traffic else moved_model) / (kern_avg_ms * 1e-3) * 1e-9 / pk["hbm_gbs"]
                                      if pk.get("hbm_gbs") else None)},
            "cpu_baseline": cpu,
        }
        print(json.dumps(out), flush=True)
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=1000)
    ap.add_argument("--warmup", type=int, default=50)
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--n", type=int, default=2048)
    ap.add_argument("--kn", type=float, default=0.1)
    ap.add_argument("--ref-n", type=int, default=512, help="grid of the bounded oracle sample")
    ap.add_argument("--cpu-steps", type=int, default=250,
                    help="oracle steps of the cpu_baseline leg (~15 s on 16 cores at 512^2)")
    ap.add_argument("--cpu-steps-single", type=int, default=16,
                    help="oracle steps of the single-thread leg (~10 s on a 512 x 128 band)")
    ap.add_argument("--developed-t", type=float, default=0.0,
                    help="advance to this time with CFL steps before the warm-up (developed-state window)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--tubes", type=int, default=4096, help="--workload sod5-batch: number of tubes")
    ap.add_argument("--workload", default="baseline", choices=sorted(WORKLOADS) + ["sod5-batch"],
                    help="baseline = BASELINE.json configs[3] (the metric); paper-* = the paper's own jet cases")
    ap.add_argument("--general-path", action="store_true",
                    help="forbid the z-symmetric kernel variant (measurement of the general one)")
    args = ap.parse_args()
    global WORKLOAD, CFL
    if args.workload == "sod5-batch":
        return run_gpu_batch5(args)
    WORKLOAD = args.workload
    CFL = WORKLOADS[WORKLOAD][1]
    if args.impl == "reference":
        run_reference(args)
    else:
        run_gpu(args)


if __name__ == "__main__":
    main()
