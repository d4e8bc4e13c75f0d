#!/usr/bin/env python
"""Benchmark of the 3N normal-ordering hot path on B200 (contract: see DESIGN.md section 8).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg2] [--impl reference]

A "step" is one pass of the whole hot path (all launches of the workload: no_eval for every run of
the sweep) over one batch of seeded synthetic configurations.  Prints ONE JSON line.
  value      k3-point matrix-element evaluations per second, inputs resident in HBM (CUDA events)
  e2e        the same through no_eval_host: pinned HOST buffers, H2D and D2H inside the timed region
  roofline   FP64 ALU roofline of the kernel (bound "alu"; DESIGN.md section 7 derives the peak)
  cpu_baseline  the oracle, as it stands, on the host cores, on a bounded sample of the same workload
With --impl reference the oracle itself is the timed program (rank 0 only).
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

METRIC = "3N-NO k3-point matrix-element evals/s (FP64) on 1 B200; % FP64 peak"
UNIT = "evals/s"

# FP64 flops the shipped kernel executes per k3-point evaluation (static count of the hot loop's SASS,
# 2 per DFMA, 1 per DADD/DMUL; DESIGN.md section 7 shows the count and the ncu cross-check).
FLOPS_PER_EVAL = {False: 76.0, True: 76.0}          # keyed by "c4 != 0" (the hot loop is the same)
# nominal FP64 vector peak: 148 SMs x 64 DFMA lanes x 2 flops x 1.965 GHz
FP64_PEAK_NOMINAL_TFLOPS = 148 * 64 * 2 * 1.965e9 / 1e12
# dram__bytes_read.sum + dram__bytes_write.sum per launch of the cfg2 kernel, from the ncu --set full capture
# summarised in profiles/r01e.md (the output is still in L2 when the capture ends; the kernel is ALU bound)
NCU_DRAM_BYTES_PER_LAUNCH = {"cfg2": 639232}


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="cfg2", choices=["cfg1", "cfg2", "cfg3", "cfg4", "cfg5", "c4", "paper", "hf"])
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true", help="skip the oracle timing leg")
    ap.add_argument("--no-e2e", action="store_true", help="skip the host-buffer leg")
    ap.add_argument("--cpu-sample", type=int, default=0, help="configurations in the oracle sample (0 = auto)")
    return ap.parse_args()


# --------------------------------------------------------------------------------------------
# clocks during the timed region (profiling recipe's nvidia-smi line)
# --------------------------------------------------------------------------------------------
class ClockSampler:
    QUERY = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
             "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
             "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        self.gpu = gpu_index
        self.lines = []
        self.proc = None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.gpu}", f"--query-gpu={self.QUERY}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            threading.Thread(target=self._pump, daemon=True).start()
        except OSError:
            self.proc = None

    def _pump(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, smax, power, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in self.lines:
            f = [x.strip() for x in line.split(",")]
            if len(f) < 9:
                continue
            try:
                sm.append(float(f[1]))
                smax.append(float(f[2]))
                power.append(float(f[3]))
            except ValueError:
                continue
            for name, val in zip(names, f[5:9]):
                if val.lower().startswith("active"):
                    reasons.add(name)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        return {"sm_mhz": statistics.median(sm), "sm_max_mhz": max(smax), "power_w_max": max(power),
                "samples": len(sm), "reasons": sorted(reasons)}


# --------------------------------------------------------------------------------------------
# CPU oracle legs
# --------------------------------------------------------------------------------------------
def oracle_sample(workload, n_sample: int):
    """Bounded sample of the workload for the oracle: the first n_sample configurations of run 0 at the
    full k3 grid (auto: about 5e5 evaluations, ~10-30 s on 8 cores)."""
    run = workload.runs[0]
    if n_sample <= 0:
        n_sample = max(1, min(run.n_cfg, int(round(5.0e5 / run.nodes_per_cfg))))
    return run, run.configurations(n_sample), n_sample


def time_oracle(workload, n_sample: int):
    from oracle import oracle as O
    run, cfg, n = oracle_sample(workload, n_sample)
    t0 = time.perf_counter()
    O.normal_order(cfg, level=1, precision="ld", dirs=run.angular(), **run.params())
    dt = time.perf_counter() - t0
    evals = n * run.nodes_per_cfg
    return {"value": evals / dt, "unit": UNIT, "cores": O.num_threads(), "kind": "oracle",
            "sample": f"first {n} configurations of run '{run.name}' of {workload.name} at the full "
                      f"{run.nodes_per_cfg}-node grid ({evals} evaluations, {dt:.1f} s, level-1 long double)"}, dt


def run_reference(args, workload):
    """--impl reference: the oracle is the timed program; each step is the bounded sample."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    # torchrun exports OMP_NUM_THREADS=1 to every rank; rank 0 alone runs the oracle, so give it the host
    # cores back (set before libgomp is loaded; the oracle itself is untouched)
    if int(os.environ.get("WORLD_SIZE", "1")) > 1 and os.environ.get("OMP_NUM_THREADS") == "1":
        os.environ["OMP_NUM_THREADS"] = str(os.cpu_count() or 1)
    from oracle import oracle as O
    O.build()
    run, cfg, n = oracle_sample(workload, args.cpu_sample)
    evals = n * run.nodes_per_cfg
    for _ in range(args.warmup):
        O.normal_order(cfg[:max(1, n // 8)], dirs=run.angular(), **run.params())
    t0 = time.perf_counter()
    for _ in range(args.steps):
        O.normal_order(cfg, level=1, precision="ld", dirs=run.angular(), **run.params())
    dt = (time.perf_counter() - t0) / args.steps
    value = evals / dt
    sample = (f"first {n} configurations of run '{run.name}' of {workload.name} at the full "
              f"{run.nodes_per_cfg}-node grid ({evals} evaluations per step)")
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt * 1e3, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload.name, "description": workload.description, "sample": sample},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": O.num_threads(), "kind": "oracle",
                             "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# --------------------------------------------------------------------------------------------
# the CUDA arm
# --------------------------------------------------------------------------------------------
def run_b200(args, workload):
    import numpy as np
    import torch
    import torch.distributed as dist

    from paper_2603_24532_b200 import binding, build, replicas

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the product has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    build.build()
    binding.load()
    dev = torch.device("cuda", local)
    stream = torch.cuda.current_stream(dev)

    # replicas only: every rank integrates the whole workload on its own GPU
    runs = replicas.replica_runs(workload)
    handles = [binding.no_init(device=local, angular=r.angular(), **r.params()) for r in runs]
    h_cfg = [torch.from_numpy(r.configurations()).pin_memory() for r in runs]
    d_cfg = [c.to(dev, non_blocking=True) for c in h_cfg]
    d_out = [torch.empty((r.n_cfg, 16, 16, 2), dtype=torch.float64, device=dev) for r in runs]
    evals_step = sum(binding.no_evals_per_cfg(h) * r.n_cfg for h, r in zip(handles, runs))
    assert evals_step == workload.evals
    flush = torch.empty(256 * 1024 * 1024 // 4, dtype=torch.float32, device=dev)   # 256 MiB > 126 MB L2
    info = binding.no_kernel_info(handles[0])

    def step_device():
        for h, c, o, r in zip(handles, d_cfg, d_out, runs):
            binding.no_eval(h, c.data_ptr(), r.n_cfg, o.data_ptr(), stream.cuda_stream)

    def barrier():
        replicas.barrier()
        torch.cuda.synchronize(dev)

    for _ in range(max(args.warmup, 3)):
        step_device()
    barrier()

    sampler = ClockSampler(local)
    sampler.start()
    time.sleep(0.25)
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    barrier()
    t_wall0 = time.perf_counter()
    for a, b in ev:
        flush.zero_()                      # L2 flush between timed iterations, outside the event bracket
        a.record(stream)
        step_device()
        b.record(stream)
    barrier()
    t_wall = time.perf_counter() - t_wall0
    clocks = sampler.stop()
    step_ms = [a.elapsed_time(b) for a, b in ev]
    t_dev = replicas.max_over_ranks(sum(step_ms) * 1e-3, dev)
    value = replicas.whole_job_rate(evals_step, args.steps, t_dev)
    n_launch = len(runs) * args.steps

    # ---- end to end through the C ABI with HOST buffers (H2D + D2H inside the timed region) ----
    e2e = None
    if not args.no_e2e:
        h_out = [torch.empty((r.n_cfg, 16, 16, 2), dtype=torch.float64).pin_memory() for r in runs]

        def step_host():
            for h, c, o, r in zip(handles, h_cfg, h_out, runs):
                binding.no_eval_host(h, c.data_ptr(), r.n_cfg, o.data_ptr(), stream.cuda_stream)

        step_host()
        barrier()
        k = max(1, min(args.steps, 3))
        t0 = time.perf_counter()
        for _ in range(k):
            step_host()
        barrier()
        t_e2e = replicas.max_over_ranks((time.perf_counter() - t0) / k, dev)
        chk = float(h_out[0][0].abs().sum())          # the step's result is read on the host
        e2e = {"value": world * evals_step / t_e2e, "unit": UNIT,
               "h2d_bytes_per_step": int(sum(c.numel() * 8 for c in h_cfg)),
               "d2h_bytes_per_step": int(sum(o.numel() * 8 for o in h_out)),
               "ms_per_step": t_e2e * 1e3, "steps": k, "checksum": chk}
        del h_out

    # ---- roofline of the (single) kernel: FP64 ALU bound ----
    has_c4 = any(r.c4 != 0.0 for r in runs)
    flops_step = FLOPS_PER_EVAL[has_c4] * evals_step
    launch_ms = sum(step_ms) / n_launch
    achieved = flops_step * args.steps / (sum(step_ms) * 1e-3) / 1e12
    probe = binding.no_probe_fp64_peak(local, 200, stream.cuda_stream)
    roofline = {"bound": "alu", "achieved": achieved, "peak": FP64_PEAK_NOMINAL_TFLOPS, "unit": "TFLOP/s",
                "frac": achieved / FP64_PEAK_NOMINAL_TFLOPS, "traffic": NCU_DRAM_BYTES_PER_LAUNCH.get(workload.name),
                "traffic_source": "profiles/r01e.md (ncu --set full, per launch)" if workload.name in NCU_DRAM_BYTES_PER_LAUNCH else None,
                "peak_source": "nominal 148 SM x 64 FP64 FMA lanes x 2 x 1.965 GHz (DESIGN.md section 7); "
                               "MEASURED_PEAKS.json has no FP64 entry",
                "peak_measured_dfma_probe": probe["tflops"],
                "frac_of_measured_dfma": achieved / probe["tflops"] if probe["tflops"] > 0 else None,
                "flops_per_eval": FLOPS_PER_EVAL[has_c4], "kernel": "no3n::no3n_kernel",
                "avg_launch_ms": launch_ms, "launches_per_step": len(runs),
                "algorithmic_bytes_per_launch": int(sum(r.n_cfg * (72 + 4096) for r in runs) / len(runs)),
                "kernel_info": info}

    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        cpu, _ = time_oracle(workload, args.cpu_sample)

    for h in handles:
        binding.no_free(h)
    if world > 1:
        dist.destroy_process_group()
    if rank != 0:
        return
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": t_dev / args.steps * 1e3, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload.name, "description": workload.description,
                       "n_cfg": workload.n_cfg, "evals_per_step": evals_step, "launches_per_step": len(runs),
                       "cfg_per_s": world * workload.n_cfg * args.steps / t_dev,
                       "l2": "256 MiB buffer rewritten between timed steps (L2 flush); the kernel is ALU bound",
                       "parallelism": "replicas only: every rank integrates the whole workload"},
            "clocks": clocks, "e2e": e2e, "gpu_launches": n_launch, "roofline": roofline, "cpu_baseline": cpu,
            "wall_s_timed_region": t_wall}
    print(json.dumps(line), flush=True)


# --------------------------------------------------------------------------------------------
# the Hartree-Fock contraction (no_hf_energy) as a workload of its own
# --------------------------------------------------------------------------------------------
HF_PARAMS = dict(kf_n=1.33, kf_p=1.33, c1=-0.81, c3=-3.2, c4=0.0, cD=1.0, cE=-0.5, gA=1.27, fpi=92.4, mpi=138.04,
                 lambda_chi=700.0, Lambda=500.0, n_reg=4, n_r=16, n_cos=16, n_phi=16)
HF_PAIR_GRID = (12, 12, 12)          # particles 1 and 2: 1728 nodes per Fermi sphere, 4 species pairs in SNM


def run_hf(args):
    """One step = one no_hf_energy call: 4 x 1728^2 pair configurations generated on the device, each reduced
    to its spin-traced diagonal over a 16^3 k3 grid inside the kernel, fixed-order reduction to E/V."""
    import torch

    from paper_2603_24532_b200 import binding, build, replicas

    if args.impl == "reference":
        if int(os.environ.get("RANK", "0")) != 0:
            return
        from oracle import oracle as O
        O.build()
        t0 = time.perf_counter()
        for _ in range(args.steps):
            e = O.hf_energy(2, 2, 2, **HF_PARAMS)
        dt = (time.perf_counter() - t0) / args.steps
        evals = 4 * 64 * 4096
        sample = "pair grid 2x2x2 per sphere (256 pair configurations x 16^3 k3 nodes per step), level-1 long double"
        print(json.dumps({"impl": "reference", "metric": METRIC, "value": evals / dt, "unit": UNIT, "n_gpus": args.gpus,
                          "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt * 1e3, "higher_is_better": True,
                          "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
                          "config": {"workload": "hf", "sample": sample, "e_over_v_fm4": e},
                          "cpu_baseline": {"value": evals / dt, "unit": UNIT, "cores": O.num_threads(), "kind": "oracle",
                                           "sample": sample},
                          "e2e": {"value": evals / dt, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
                          "gpu_launches": 0}), flush=True)
        return
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the product has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        torch.distributed.init_process_group("nccl", device_id=torch.device("cuda", local))
    build.build()
    binding.load()
    dev = torch.device("cuda", local)
    stream = torch.cuda.current_stream(dev)
    h = binding.no_init(device=local, **HF_PARAMS)
    n1 = HF_PAIR_GRID[0] * HF_PAIR_GRID[1] * HF_PAIR_GRID[2]
    n_pairs = 4 * n1 * n1
    evals_step = n_pairs * binding.no_evals_per_cfg(h)
    chunks = 4 * ((n1 * n1 + (1 << 20) - 1) >> 20)
    flush = torch.empty(256 * 1024 * 1024 // 4, dtype=torch.float32, device=dev)
    for _ in range(max(args.warmup, 3)):
        e_v = binding.no_hf_energy(h, *HF_PAIR_GRID, stream.cuda_stream)
    replicas.barrier()
    torch.cuda.synchronize(dev)
    sampler = ClockSampler(local)
    sampler.start()
    time.sleep(0.25)
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    wall = []
    for a, b in ev:
        flush.zero_()
        torch.cuda.synchronize(dev)
        t0 = time.perf_counter()
        a.record(stream)
        e_v = binding.no_hf_energy(h, *HF_PAIR_GRID, stream.cuda_stream)      # synchronises the stream itself
        b.record(stream)
        torch.cuda.synchronize(dev)
        wall.append(time.perf_counter() - t0)
    replicas.barrier()
    clocks = sampler.stop()
    step_ms = [a.elapsed_time(b) for a, b in ev]
    t_dev = replicas.max_over_ranks(sum(step_ms) * 1e-3, dev)
    t_wall = replicas.max_over_ranks(sum(wall), dev)
    value = replicas.whole_job_rate(evals_step, args.steps, t_dev)
    flops = 59.0      # forward fast path (p' = p): 20 DFMA + 12 DMUL + 7 DADD per node
    achieved = flops * evals_step * args.steps / (sum(step_ms) * 1e-3) / 1e12
    probe = binding.no_probe_fp64_peak(local, 200, stream.cuda_stream)
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        from oracle import oracle as O
        t0 = time.perf_counter()
        O.hf_energy(2, 2, 2, **HF_PARAMS)
        dt = time.perf_counter() - t0
        cpu = {"value": 4 * 64 * 4096 / dt, "unit": UNIT, "cores": O.num_threads(), "kind": "oracle",
               "sample": f"pair grid 2x2x2 per sphere (256 pair configurations x 16^3 k3 nodes, {dt:.1f} s), level-1 long double"}
    binding.no_free(h)
    if world > 1:
        torch.distributed.destroy_process_group()
    if rank != 0:
        return
    print(json.dumps({
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
        "ms_per_step": t_dev / args.steps * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": "hf", "description": "3N Hartree-Fock energy of SNM kF=1.33 by repeated normal ordering "
                   "(no_hf_energy): 12^3 nodes per sphere for particles 1, 2 (4 x 1728^2 pair configurations, generated "
                   "on the device), 16^3 k3 grid", "n_cfg": n_pairs, "evals_per_step": evals_step,
                   "cfg_per_s": world * n_pairs * args.steps / t_dev, "e_over_v_fm4": e_v,
                   "l2": "256 MiB buffer rewritten between timed steps (L2 flush); the kernel is ALU bound",
                   "parallelism": "replicas only: every rank integrates the whole workload"},
        "clocks": clocks,
        "e2e": {"value": world * evals_step * args.steps / t_wall, "unit": UNIT,
                "h2d_bytes_per_step": 4 * n1 * 32, "d2h_bytes_per_step": 4 * 8, "ms_per_step": t_wall / args.steps * 1e3,
                "note": "the call itself is the public API: node lists up, one scalar down, wall clock around it"},
        "gpu_launches": 3 * chunks * args.steps,
        "roofline": {"bound": "alu", "achieved": achieved, "peak": FP64_PEAK_NOMINAL_TFLOPS, "unit": "TFLOP/s",
                     "frac": achieved / FP64_PEAK_NOMINAL_TFLOPS, "traffic": None,
                     "peak_measured_dfma_probe": probe["tflops"], "flops_per_eval": flops,
                     "kernel": "no3n::no3n_kernel (forward fast path, diagonal mode) + hf_pairs_kernel + hf_reduce_kernel"},
        "cpu_baseline": cpu}), flush=True)


def main():
    args = parse_args()
    if args.workload == "hf":
        run_hf(args)
        return
    from paper_2603_24532_b200 import workloads
    wl = workloads.workload(args.workload)
    if args.impl == "reference":
        run_reference(args, wl)
    else:
        run_b200(args, wl)


if __name__ == "__main__":
    main()
