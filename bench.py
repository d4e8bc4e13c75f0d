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

# nominal FP64 vector peak: 148 SMs x 64 DFMA lanes x 2 flops x 1.965 GHz
FP64_PEAK_NOMINAL_TFLOPS = 148 * 64 * 2 * 1.965e9 / 1e12
# dram__bytes_read.sum + dram__bytes_write.sum per launch (mean over the launches of one step) of the workload's
# kernel, from the ncu capture named beside it (profiles/); None = no capture of that workload exists
NCU_DRAM_BYTES_PER_LAUNCH = {"cfg5": 1655888896, "trace5": 5376942696}
NCU_DRAM_SOURCE = {"cfg5": "profiles/r02a.md (r02a_cfg5_dram.csv: all six launches of one cfg5 step, 9.94 GB of DRAM "
                           "traffic against 9.83 GB algorithmic: 4.4 GB of output per 2^20-configuration launch cannot stay in the 126 MB L2)",
                   "trace5": "profiles/r02b.md (ncu --set full of one launch: 5.3688 GB read + 0.0082 GB written against 5.3729 GB "
                             "algorithmic)"}


def flops_per_eval(n_reg: int, regulated: bool, forward: bool = False) -> float:
    """FP64 flops the shipped kernel executes per k3-point evaluation, by kernel variant: static count of the
    hot loop body (no3n::nodes; 2 per DFMA, 1 per DADD/DMUL; DESIGN.md section 7 shows the count and the ncu
    cross-check).  Regulated, exponent n: 22 + (n - 1) DFMA, 16 DMUL, 10 DADD (n = 4: 25/16/10 = 76 flops);
    unregulated: 15/14/9; the forward variant (p' = p) drops 5 DFMA, 4 DMUL, 3 DADD."""
    if regulated:
        fma, mul, add = 22 + (n_reg - 1), 16, 10
    else:
        fma, mul, add = 15, 14, 9
    if forward:
        fma, mul, add = fma - 5, mul - 4, add - 3
    return float(2 * fma + mul + add)


def run_flops(run) -> float:
    return flops_per_eval(run.n_reg, run.Lambda > 0)


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="cfg5", choices=["cfg1", "cfg2", "cfg3", "cfg4", "cfg5", "c4", "paper", "hf", "trace5", "trace6"])
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true", help="skip the oracle timing leg")
    ap.add_argument("--no-e2e", action="store_true", help="skip the host-buffer leg")
    ap.add_argument("--no-per-config", action="store_true", help="skip the short runs of the other BASELINE configs")
    ap.add_argument("--no-per-workload", action="store_true",
                    help="skip the short legs of the section-8(f) workloads (paper quadrature, hf, trace5) on the default line")
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
def oracle_sample(workload, n_sample: int, target_evals: float):
    """Bounded sample of the workload for the oracle: the first n_sample configurations of run 0 at the
    full k3 grid (auto: about target_evals evaluations, at least one configuration per host core so that the
    OpenMP loop over configurations uses every core)."""
    from oracle import oracle as O
    run = workload.runs[0]
    if n_sample <= 0:
        n_sample = max(O.num_threads(), int(round(target_evals / run.nodes_per_cfg)))
    n_sample = max(1, min(run.n_cfg, n_sample))
    return run, run.configurations(n_sample), n_sample


ORACLE_KIND = "oracle (level 1, f64 instantiation; the parity reference is the long-double one)"


def time_oracle(workload, n_sample: int):
    """cpu_baseline: the oracle as it stands (level 1, double), about 10-20 s on the box's host cores."""
    from oracle import oracle as O
    run, cfg, n = oracle_sample(workload, n_sample, 8.0e6)
    t0 = time.perf_counter()
    O.normal_order(cfg, level=1, precision="f64", dirs=run.angular(), **run.params())
    dt = time.perf_counter() - t0
    evals = n * run.nodes_per_cfg
    return {"value": evals / dt, "unit": UNIT, "cores": O.num_threads(), "kind": ORACLE_KIND,
            "sample": f"first {n} configurations of run '{run.name}' of {workload.name} at the full "
                      f"{run.nodes_per_cfg}-node grid ({evals} evaluations, {dt:.1f} s)"}, dt


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
    run, cfg, n = oracle_sample(workload, args.cpu_sample, 2.5e6)
    evals = n * run.nodes_per_cfg
    for _ in range(args.warmup):
        O.normal_order(cfg[:max(1, n // 8)], level=1, precision="f64", dirs=run.angular(), **run.params())
    t0 = time.perf_counter()
    for _ in range(args.steps):
        O.normal_order(cfg, level=1, precision="f64", dirs=run.angular(), **run.params())
    dt = (time.perf_counter() - t0) / args.steps
    value = evals / dt
    sample = (f"first {n} configurations of run '{run.name}' of {workload.name} at the full "
              f"{run.nodes_per_cfg}-node grid ({evals} evaluations per step)")
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt * 1e3, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload.name, "description": workload.description, "sample": sample},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": O.num_threads(), "kind": ORACLE_KIND,
                             "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# --------------------------------------------------------------------------------------------
# the CUDA arm
# --------------------------------------------------------------------------------------------
class DeviceWorkload:
    """A workload resident on the device: one handle, one configuration array and one output array per run."""

    def __init__(self, workload, local, dev, pinned_inputs=False):
        import torch

        from paper_2603_24532_b200 import binding, replicas
        self.binding = binding
        self.workload = workload
        # replicas only: every rank integrates the whole workload on its own GPU
        self.runs = replicas.replica_runs(workload)
        self.handles = [binding.no_init(device=local, angular=r.angular(), **r.params()) for r in self.runs]
        self.h_cfg = [torch.from_numpy(r.configurations()) for r in self.runs]
        if pinned_inputs:
            self.h_cfg = [c.pin_memory() for c in self.h_cfg]
        self.d_cfg = [c.to(dev, non_blocking=True) for c in self.h_cfg]
        self.d_out = [torch.empty((r.n_cfg, 16, 16, 2), dtype=torch.float64, device=dev) for r in self.runs]
        self.evals_step = sum(binding.no_evals_per_cfg(h) * r.n_cfg for h, r in zip(self.handles, self.runs))
        assert self.evals_step == workload.evals
        self.flops_step = sum(run_flops(r) * r.evals for r in self.runs)

    def step(self, stream):
        for h, c, o, r in zip(self.handles, self.d_cfg, self.d_out, self.runs):
            self.binding.no_eval(h, c.data_ptr(), r.n_cfg, o.data_ptr(), stream.cuda_stream)

    def close(self):
        for h in self.handles:
            self.binding.no_free(h)
        self.handles = []
        self.d_cfg = self.d_out = self.h_cfg = None


def timed_steps(dw, stream, dev, flush, steps, warmup, barrier):
    """`warmup` untimed steps, then `steps` timed ones: CUDA events on the launching stream around each step,
    the L2 flushed (256 MiB rewritten) before each, outside the event bracket.  Returns the per-step ms."""
    import torch
    for _ in range(warmup):
        dw.step(stream)
    barrier()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    for a, b in ev:
        flush.zero_()
        a.record(stream)
        dw.step(stream)
        b.record(stream)
    barrier()
    return [a.elapsed_time(b) for a, b in ev]


def small_batch_rates(dw, dev):
    """Small transactions (cfg1: 256 configurations per launch, the paper's per-diagram transaction size):
    launches back to back on one stream, and the same launches spread over 4 streams and replayed as ONE CUDA graph
    (many host threads sharing the GPU through streams, without the host-side launch cost)."""
    import torch
    h, c, o, r = dw.handles[0], dw.d_cfg[0], dw.d_out[0], dw.runs[0]
    evals = dw.binding.no_evals_per_cfg(h) * r.n_cfg
    reps = 64
    main = torch.cuda.current_stream(dev)
    outs = [torch.empty_like(o) for _ in range(4)]
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    for _ in range(8):
        dw.binding.no_eval(h, c.data_ptr(), r.n_cfg, o.data_ptr(), main.cuda_stream)
    a.record(main)
    for _ in range(reps):
        dw.binding.no_eval(h, c.data_ptr(), r.n_cfg, o.data_ptr(), main.cuda_stream)
    b.record(main)
    torch.cuda.synchronize(dev)
    serial = evals * reps / (a.elapsed_time(b) * 1e-3)
    streams = [torch.cuda.Stream(dev) for _ in range(4)]
    g = torch.cuda.CUDAGraph()
    cap = torch.cuda.Stream(dev)
    with torch.cuda.stream(cap):
        with torch.cuda.graph(g, stream=cap):
            for k in range(reps):
                st = streams[k % 4]
                st.wait_stream(cap)
                dw.binding.no_eval(h, c.data_ptr(), r.n_cfg, outs[k % 4].data_ptr(), st.cuda_stream)
            for st in streams:
                cap.wait_stream(st)
    for _ in range(3):
        g.replay()
    torch.cuda.synchronize(dev)
    a.record(main)
    for _ in range(4):
        g.replay()
    b.record(main)
    torch.cuda.synchronize(dev)
    graph = evals * reps * 4 / (a.elapsed_time(b) * 1e-3)
    assert torch.equal(outs[0], o)
    return {"back_to_back_one_stream_evals_per_s": serial, "graph_4_streams_evals_per_s": graph, "launches": reps}


def build_once(world: int, local: int):
    """compile libno3n.so if it is stale: local rank 0 alone (the other ranks of the node wait), so that N ranks never
    run nvcc on the same output file"""
    import torch.distributed as dist

    from paper_2603_24532_b200 import binding, build
    if world > 1:
        if local == 0:
            build.build()
        dist.barrier()
    else:
        build.build()
    binding.load()


def run_b200(args, workload):
    import torch
    import torch.distributed as dist

    from paper_2603_24532_b200 import binding, build, replicas, workloads

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the product has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    build_once(world, local)
    dev = torch.device("cuda", local)
    stream = torch.cuda.current_stream(dev)

    dw = DeviceWorkload(workload, local, dev, pinned_inputs=not args.no_e2e)
    runs, handles, evals_step = dw.runs, dw.handles, dw.evals_step
    flush = torch.empty(256 * 1024 * 1024 // 4, dtype=torch.float32, device=dev)   # 256 MiB > 126 MB L2
    info = binding.no_kernel_info(handles[0])

    def barrier():
        replicas.barrier()
        torch.cuda.synchronize(dev)

    warmup = max(args.warmup, 3)
    for _ in range(warmup):
        dw.step(stream)
    barrier()
    sampler = ClockSampler(local)
    sampler.start()
    time.sleep(0.25)
    t_wall0 = time.perf_counter()
    step_ms = timed_steps(dw, stream, dev, flush, args.steps, 0, barrier)
    t_wall = time.perf_counter() - t_wall0
    clocks = sampler.stop()
    t_dev = replicas.max_over_ranks(sum(step_ms) * 1e-3, dev)
    value = replicas.whole_job_rate(evals_step, args.steps, t_dev)
    n_launch = len(runs) * args.steps

    # ---- the same step writing the packed, symmetry-reduced form (no_eval_packed; device resident, not the headline) ----
    packed_dev = None
    if world == 1:
        pk = []
        for h, r in zip(handles, runs):
            fmt = binding.NO_PACK_ISOSPIN if binding.no_packed_doubles(h, binding.NO_PACK_ISOSPIN) else binding.NO_PACK_CHARGE
            pk.append((fmt, torch.empty((r.n_cfg, binding.no_packed_doubles(h, fmt)), dtype=torch.float64, device=dev)))

        def step_packed():
            for h, c, r, (fmt, o) in zip(handles, dw.d_cfg, runs, pk):
                binding.no_eval_packed(h, fmt, c.data_ptr(), r.n_cfg, o.data_ptr(), stream.cuda_stream)

        step_packed()
        kp = max(1, min(args.steps, 3))
        evp = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(kp)]
        for a, b in evp:
            flush.zero_()
            a.record(stream)
            step_packed()
            b.record(stream)
        torch.cuda.synchronize(dev)
        ms = sum(a.elapsed_time(b) for a, b in evp)
        packed_dev = {"evals_per_s": evals_step * kp / (ms * 1e-3), "steps": kp,
                      "bytes_out_per_step": int(sum(o.numel() * 8 for _, o in pk)),
                      "api": "no_eval_packed (isospin form where kF_n = kF_p, charge form otherwise), outputs resident in HBM"}
        del pk

    # ---- end to end through the C ABI with HOST buffers (H2D + D2H inside the timed region) ----
    # e2e: no_eval_host_packed, the symmetry-reduced form the paper describes (isospin form for runs
    # with kF_n = kF_p, charge-conserving form otherwise; the full matrix follows by an index map, no_unpack);
    # e2e_full_matrices: no_eval_host, all 256 entries of every matrix over PCIe.
    def e2e_leg(packed: bool):
        fmts = []
        for h in handles:
            if not packed:
                fmts.append((0, 512))
            elif binding.no_packed_doubles(h, binding.NO_PACK_ISOSPIN):
                fmts.append((binding.NO_PACK_ISOSPIN, binding.no_packed_doubles(h, binding.NO_PACK_ISOSPIN)))
            else:
                fmts.append((binding.NO_PACK_CHARGE, binding.no_packed_doubles(h, binding.NO_PACK_CHARGE)))
        h_out = [torch.empty((r.n_cfg, pd), dtype=torch.float64, pin_memory=True) for r, (_, pd) in zip(runs, fmts)]

        def step_host():
            for h, c, o, r, (fmt, _) in zip(handles, dw.h_cfg, h_out, runs, fmts):
                if fmt:
                    binding.no_eval_host_packed(h, fmt, c.data_ptr(), r.n_cfg, o.data_ptr(), stream.cuda_stream)
                else:
                    binding.no_eval_host(h, c.data_ptr(), r.n_cfg, o.data_ptr(), stream.cuda_stream)

        step_host()
        barrier()
        k = max(1, min(args.steps, 5))
        t0 = time.perf_counter()
        for _ in range(k):
            step_host()
        barrier()
        t_e2e = replicas.max_over_ranks((time.perf_counter() - t0) / k, dev)
        chk = float(h_out[0][0].abs().sum())          # the step's result is read on the host
        names = {0: "full 16x16", binding.NO_PACK_CHARGE: "NO_PACK_CHARGE (96 entries)",
                 binding.NO_PACK_ISOSPIN: "NO_PACK_ISOSPIN (32 entries)"}
        return {"value": world * evals_step / t_e2e, "unit": UNIT,
                "h2d_bytes_per_step": int(sum(c.numel() * 8 for c in dw.h_cfg)),
                "d2h_bytes_per_step": int(sum(o.numel() * 8 for o in h_out)),
                "ms_per_step": t_e2e * 1e3, "steps": k, "checksum": chk,
                "api": ("no_eval_host_packed" if packed else "no_eval_host") + " (pinned host buffers); result form per run: "
                       + ", ".join(sorted({names[f] for f, _ in fmts}))}

    e2e = e2e_full = None
    if not args.no_e2e:
        e2e = e2e_leg(True)
        e2e_full = e2e_leg(False)

    # ---- roofline of the (single) kernel: FP64 ALU bound ----
    launch_ms = sum(step_ms) / n_launch
    achieved = dw.flops_step * args.steps / (sum(step_ms) * 1e-3) / 1e12
    probe = binding.no_probe_fp64_peak(local, 200, stream.cuda_stream)
    per_run_flops = sorted({run_flops(r) for r in runs})
    roofline = {"bound": "alu", "achieved": achieved, "peak": FP64_PEAK_NOMINAL_TFLOPS, "unit": "TFLOP/s",
                "frac": achieved / FP64_PEAK_NOMINAL_TFLOPS, "traffic": NCU_DRAM_BYTES_PER_LAUNCH.get(workload.name),
                "traffic_source": NCU_DRAM_SOURCE.get(workload.name),
                "peak_source": "nominal 148 SM x 64 FP64 FMA lanes x 2 x 1.965 GHz (DESIGN.md section 7); "
                               "MEASURED_PEAKS.json has no FP64 entry, the in-run DFMA probe is the measured figure",
                "peak_measured_dfma_probe": probe["tflops"],
                "frac_of_measured_dfma": achieved / probe["tflops"] if probe["tflops"] > 0 else None,
                "flops_per_eval": dw.flops_step / evals_step, "flops_per_eval_by_variant": per_run_flops,
                "kernel": "no3n::no3n_kernel", "avg_launch_ms": launch_ms, "launches_per_step": len(runs),
                "algorithmic_bytes_per_launch": int(sum(r.n_cfg * (72 + 4096) for r in runs) / len(runs)),
                "kernel_info": info}
    small = small_batch_rates(dw, dev) if workload.name == "cfg1" and world == 1 else None
    dw.close()

    # ---- the other BASELINE configs, a few steps each in the same run (not the headline) ----
    per_config = None
    if world == 1 and not args.no_per_config:
        per_config = {}
        for name in ("cfg1", "cfg2", "cfg3", "cfg4", "cfg5"):
            if name == workload.name:
                continue
            if name == "cfg5" and args.workload != "cfg5":
                continue                                           # 2.8 s per step: only as the headline
            wl = workloads.workload(name)
            d2 = DeviceWorkload(wl, local, dev)
            ms = timed_steps(d2, stream, dev, flush, 3, 3, barrier)
            rate = wl.evals * len(ms) / (sum(ms) * 1e-3)
            fl = d2.flops_step / wl.evals
            extra = small_batch_rates(d2, dev) if name == "cfg1" else None
            per_config[name] = {"small_transactions": extra, "evals_per_s": rate, "cfg_per_s": wl.n_cfg * len(ms) / (sum(ms) * 1e-3),
                                "ms_per_step": sum(ms) / len(ms), "steps": len(ms), "flops_per_eval": fl,
                                "frac": rate * fl / 1e12 / FP64_PEAK_NOMINAL_TFLOPS}
            d2.close()
            del d2
            torch.cuda.empty_cache()

    # ---- the section-8(f) workloads on the same line: short legs, each the code path of `bench.py --workload X` ----
    per_workload = None
    if world == 1 and workload.name == "cfg5" and not args.no_per_workload:
        del flush
        torch.cuda.empty_cache()
        per_workload = per_workload_legs()

    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        cpu, _ = time_oracle(workload, args.cpu_sample)

    if world > 1:
        dist.destroy_process_group()
    if rank != 0:
        return
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": warmup, "ms_per_step": t_dev / args.steps * 1e3, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload.name, "description": workload.description,
                       "n_cfg": workload.n_cfg, "evals_per_step": evals_step, "launches_per_step": len(runs),
                       "cfg_per_s": world * workload.n_cfg * args.steps / t_dev,
                       "l2": "256 MiB buffer rewritten between timed steps (L2 flush); the kernel is ALU bound",
                       "parallelism": "replicas only: every rank integrates the whole workload",
                       "per_config": per_config, "per_workload": per_workload, "small_transactions": small,
                       "packed_output": packed_dev},
            "clocks": clocks, "e2e": e2e, "e2e_full_matrices": e2e_full, "gpu_launches": n_launch, "roofline": roofline, "cpu_baseline": cpu,
            "wall_s_timed_region": t_wall}
    print(json.dumps(line), flush=True)


def per_workload_legs():
    """Short legs (3 timed steps after 3 warm-up steps; the trace leg keeps its 20 one-millisecond launches) of the
    workloads of SURVEY.md 8(f): the paper's quadrature (f2), the Hartree-Fock contraction (f1,
    PAPER.md:188) and the fifth-order trace with unpacked and packed input (f4).  Each leg IS
    `bench.py --workload X` (same L2 flush, CUDA-event timing, clock sampling, e2e through the public API), run as a
    child process on the same GPU after this process has released its buffers, so the default line carries its
    roofline object, e2e and clocks.  A leg that fails is reported as {"error": ...}; it never fails the line."""
    legs = {}
    keep_roofline = ("bound", "achieved", "peak", "unit", "frac", "flops_per_eval", "useful_bytes_per_sample",
                     "frac_all_bytes_read", "hbm_gbs_all_bytes_read", "limiter", "avg_launch_ms", "kernel",
                     "peak_measured_dfma_probe", "fp64_tflops")
    for name in ("paper", "hf", "trace5"):
        cmd = [sys.executable, os.path.abspath(__file__), "--workload", name, "--steps", "3", "--warmup", "3",
               "--no-cpu-baseline", "--no-per-config", "--no-per-workload"]
        t0 = time.perf_counter()
        try:
            r = subprocess.run(cmd, capture_output=True, text=True, timeout=900, cwd=ROOT)
            rows = [l for l in r.stdout.splitlines() if l.startswith("{")]
            if r.returncode != 0 or not rows:
                legs[name] = {"error": f"rc {r.returncode}: {r.stderr.strip()[-300:]}"}
                continue
            d = json.loads(rows[-1])
        except (subprocess.TimeoutExpired, OSError, ValueError) as exc:
            legs[name] = {"error": repr(exc)[:300]}
            continue
        rf = d.get("roofline") or {}
        e2e = d.get("e2e") or {}
        legs[name] = {"metric": d["metric"], "value": d["value"], "unit": d["unit"], "ms_per_step": d["ms_per_step"],
                      "steps": d["steps"], "warmup": d["warmup"], "gpu_launches": d["gpu_launches"],
                      "roofline": {k: rf[k] for k in keep_roofline if k in rf},
                      "e2e": {k: e2e[k] for k in ("value", "unit", "h2d_bytes_per_step", "d2h_bytes_per_step", "ms_per_step", "api")
                              if k in e2e},
                      "clocks": d.get("clocks"), "description": d["config"].get("description"),
                      "wall_s": time.perf_counter() - t0}
        if name == "trace5" and "packed_input" in rf:
            pk, peak = rf["packed_input"], rf["peak"]
            legs["trace5_packed_input"] = {
                "metric": d["metric"], "value": pk["samples_per_s"], "unit": d["unit"], "ms_per_step": pk["avg_launch_ms"],
                "steps": 10, "warmup": 3, "gpu_launches": 10,
                "roofline": {"bound": "hbm", "achieved": pk["hbm_gbs"], "peak": peak, "unit": "GB/s", "frac": pk["hbm_gbs"] / peak,
                             "bytes_per_sample": pk["bytes_per_sample"], "avg_launch_ms": pk["avg_launch_ms"],
                             "kernel": "trace_kernel (no_trace_eval_packed, NO_PACK_CHARGE input)", "limiter": rf.get("limiter")},
                "e2e": None, "clocks": d.get("clocks"), "description": pk["api"]}
    return legs


# --------------------------------------------------------------------------------------------
# the Hartree-Fock contraction (no_hf_energy) as a workload of its own
# --------------------------------------------------------------------------------------------
HF_PARAMS = dict(kf_n=1.33, kf_p=1.33, c1=-0.81, c3=-3.2, c4=0.0, cD=1.0, cE=-0.5, gA=1.27, fpi=92.4, mpi=138.04,
                 lambda_chi=700.0, Lambda=500.0, n_reg=4, n_r=16, n_cos=16, n_phi=16)
HF_PAIR_GRID = (12, 12, 12)          # particles 1 and 2: 1728 nodes per Fermi sphere, 4 species pairs in SNM
# Both arms count the SAME unit of work: (pair configurations of ONE pair grid) x (k3 nodes), i.e. what one energy
# needs once the coinciding isospin pair grids of kF_n = kF_p are integrated once (as no_hf_energy does).  The oracle
# as it stands loops over all four (t1, t2) grids; that redundancy is its own and is not credited.  Both in f64.
HF_CPU_EVALS = 8 * 8 * 4096
HF_CPU_SAMPLE = ("pair grid 2x2x2 per sphere: 64 pair configurations x 16^3 k3 nodes counted per step (the oracle evaluates "
                 "them once per isospin pair, 4x, uncredited), level-1 oracle in f64")


def run_hf(args):
    """One step = one no_hf_energy call: 1728^2 pair configurations generated on the device, each reduced
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
            e = O.hf_energy(2, 2, 2, precision="f64", **HF_PARAMS)
        dt = (time.perf_counter() - t0) / args.steps
        evals = HF_CPU_EVALS
        sample = HF_CPU_SAMPLE
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
    build_once(world, local)
    dev = torch.device("cuda", local)
    stream = torch.cuda.current_stream(dev)
    h = binding.no_init(device=local, **HF_PARAMS)
    n1 = HF_PAIR_GRID[0] * HF_PAIR_GRID[1] * HF_PAIR_GRID[2]
    # kF_n = kF_p: the four (t1, t2) pair grids coincide and the library integrates the pair grid once
    n_pairs = n1 * n1
    evals_step = n_pairs * binding.no_evals_per_cfg(h)
    chunks = (n1 * n1 + (1 << 20) - 1) >> 20
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
    # forward fast path (p' = p): 20 DFMA + 12 DMUL + 7 DADD per node = 59 flop (tests/test_sass_flops.py reads the count from the binary)
    flops = flops_per_eval(HF_PARAMS["n_reg"], HF_PARAMS["Lambda"] > 0, forward=True)
    achieved = flops * evals_step * args.steps / (sum(step_ms) * 1e-3) / 1e12
    probe = binding.no_probe_fp64_peak(local, 200, stream.cuda_stream)
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        from oracle import oracle as O
        t0 = time.perf_counter()
        O.hf_energy(2, 2, 2, precision="f64", **HF_PARAMS)
        dt = time.perf_counter() - t0
        cpu = {"value": HF_CPU_EVALS / dt, "unit": UNIT, "cores": O.num_threads(), "kind": "oracle",
               "sample": f"{HF_CPU_SAMPLE} ({dt:.1f} s)"}
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
                   "(no_hf_energy): 12^3 nodes per sphere for particles 1, 2 (1728^2 pair configurations, generated "
                   "on the device; since kF_n = kF_p the four isospin pair grids coincide and 1728^2 are integrated), 16^3 k3 grid", "n_cfg": n_pairs, "evals_per_step": evals_step,
                   "cfg_per_s": world * n_pairs * args.steps / t_dev, "e_over_v_fm4": e_v,
                   "l2": "256 MiB buffer rewritten between timed steps (L2 flush); the kernel is ALU bound",
                   "parallelism": "replicas only: every rank integrates the whole workload"},
        "clocks": clocks,
        "e2e": {"value": world * evals_step * args.steps / t_wall, "unit": UNIT,
                "h2d_bytes_per_step": n1 * 32, "d2h_bytes_per_step": 8, "ms_per_step": t_wall / args.steps * 1e3,
                "note": "the call itself is the public API: node lists up, one scalar down, wall clock around it"},
        "gpu_launches": 3 * chunks * args.steps,
        "roofline": {"bound": "alu", "achieved": achieved, "peak": FP64_PEAK_NOMINAL_TFLOPS, "unit": "TFLOP/s",
                     "frac": achieved / FP64_PEAK_NOMINAL_TFLOPS, "traffic": None,
                     "peak_measured_dfma_probe": probe["tflops"], "flops_per_eval": flops,
                     "kernel": "no3n::no3n_kernel (forward fast path, diagonal mode) + hf_pairs_kernel + hf_reduce_kernel"},
        "cpu_baseline": cpu}), flush=True)


# --------------------------------------------------------------------------------------------
# the spin-isospin trace (no_trace_eval) as a workload of its own
# --------------------------------------------------------------------------------------------
TRACE_BENCH = dict(n_vertex=5, n_sample=1 << 18, seed=7)      # fifth-order ring, 5.4 GB of vertex matrices (> L2)
TRACE_BENCHES = {"trace5": TRACE_BENCH,
                 "trace6": dict(n_vertex=6, n_sample=1 << 17, seed=7)}   # sixth order (4^12 labels per sample), 3.2 GB
TRACE_METRIC = "spin-isospin trace samples/s (ring diagram, FP64 complex) on 1 B200"


def hbm_peak_gbs():
    """measured HBM copy bandwidth of this pool's B200s (driver-written MEASURED_PEAKS.json), else the guide's fallback"""
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except (OSError, KeyError, ValueError):
        return 6650.0, "fallback (B200_PROFILING.md: 6.65 TB/s)"


def run_trace(args):
    """One step = one no_trace_eval launch over 2^18 samples of 5 vertex matrices (20 KiB per sample, read once)."""
    from paper_2603_24532_b200 import trace_workloads as TW
    spec = TRACE_BENCHES[args.workload]
    n, n_sample = spec["n_vertex"], spec["n_sample"]
    topo = TW.ring(n)
    labels = 4 ** (2 * n)
    if args.impl == "reference":
        if int(os.environ.get("RANK", "0")) != 0:
            return
        if int(os.environ.get("WORLD_SIZE", "1")) > 1 and os.environ.get("OMP_NUM_THREADS") == "1":
            os.environ["OMP_NUM_THREADS"] = str(os.cpu_count() or 1)
        from oracle import trace as T
        T.build()
        m = args.cpu_sample or (256 if n <= 5 else 32)
        V = TW.vertex_matrices(m, n, seed=spec["seed"])
        for _ in range(args.warmup):
            T.trace_bruteforce(topo, V[:16])
        t0 = time.perf_counter()
        for _ in range(args.steps):
            T.trace_bruteforce(topo, V)
        dt = (time.perf_counter() - t0) / args.steps
        sample = f"first {m} samples of the workload, brute-force sum over all 4^{2 * n} label configurations each"
        print(json.dumps({"impl": "reference", "metric": TRACE_METRIC, "value": m / dt, "unit": "samples/s",
                          "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt * 1e3,
                          "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
                          "config": {"workload": args.workload, "sample": sample},
                          "cpu_baseline": {"value": m / dt, "unit": "samples/s", "cores": os.cpu_count(), "kind": "oracle (brute force)",
                                           "sample": sample},
                          "e2e": {"value": m / dt, "unit": "samples/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
                          "gpu_launches": 0}), flush=True)
        return
    import torch

    from paper_2603_24532_b200 import binding, build, replicas, workloads
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the product has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        torch.distributed.init_process_group("nccl", device_id=torch.device("cuda", local))
    build_once(world, local)
    dev = torch.device("cuda", local)
    stream = torch.cuda.current_stream(dev)
    # the vertices are charge conserving (as no_eval output is): the plan skips the structurally zero blocks
    plan = binding.no_trace_init(topo, local, binding.NO_TRACE_CHARGE_CONSERVING)
    info = binding.no_trace_info(plan, n)
    V = TW.vertex_matrices(n_sample, n, seed=spec["seed"])
    d_V = torch.from_numpy(V).to(dev)
    d_out = torch.empty((n_sample,), dtype=torch.complex128, device=dev)
    flush = torch.empty(256 * 1024 * 1024 // 4, dtype=torch.float32, device=dev)

    def barrier():
        replicas.barrier()
        torch.cuda.synchronize(dev)

    warmup = max(args.warmup, 3)
    for _ in range(warmup):
        binding.no_trace_eval(plan, d_V.data_ptr(), n_sample, d_out.data_ptr(), stream.cuda_stream)
    barrier()
    sampler = ClockSampler(local)
    sampler.start()
    time.sleep(0.25)
    steps = max(args.steps, 20)
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    for a, b in ev:
        flush.zero_()
        a.record(stream)
        binding.no_trace_eval(plan, d_V.data_ptr(), n_sample, d_out.data_ptr(), stream.cuda_stream)
        b.record(stream)
    barrier()
    time.sleep(0.25)
    clocks = sampler.stop()
    step_ms = [a.elapsed_time(b) for a, b in ev]
    t_dev = replicas.max_over_ranks(sum(step_ms) * 1e-3, dev)
    value = replicas.whole_job_rate(n_sample, steps, t_dev)
    # the same launch with a plan for arbitrary (dense) vertex matrices, for comparison
    plan_d = binding.no_trace_init(topo, local, 0)
    for _ in range(3):
        binding.no_trace_eval(plan_d, d_V.data_ptr(), n_sample, d_out.data_ptr(), stream.cuda_stream)
    ed = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(5)]
    for a, b in ed:
        flush.zero_()
        a.record(stream)
        binding.no_trace_eval(plan_d, d_V.data_ptr(), n_sample, d_out.data_ptr(), stream.cuda_stream)
        b.record(stream)
    torch.cuda.synchronize(dev)
    dense_rate = n_sample * len(ed) / (sum(a.elapsed_time(b) for a, b in ed) * 1e-3)
    binding.no_trace_free(plan_d)
    # the same launch reading the vertices in the packed form no_eval_packed writes (1536 B per vertex)
    d_P = torch.from_numpy(TW.pack_charge(V)).to(dev)
    d_out_p = torch.empty_like(d_out)
    for _ in range(3):
        binding.no_trace_eval_packed(plan, binding.NO_PACK_CHARGE, d_P.data_ptr(), n_sample, d_out_p.data_ptr(), stream.cuda_stream)
    ep = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(10)]
    for a, b in ep:
        flush.zero_()
        a.record(stream)
        binding.no_trace_eval_packed(plan, binding.NO_PACK_CHARGE, d_P.data_ptr(), n_sample, d_out_p.data_ptr(), stream.cuda_stream)
        b.record(stream)
    binding.no_trace_eval(plan, d_V.data_ptr(), n_sample, d_out.data_ptr(), stream.cuda_stream)
    torch.cuda.synchronize(dev)
    assert torch.equal(d_out_p, d_out)                   # same plan, same bits from either input form
    packed_ms = sum(a.elapsed_time(b) for a, b in ep) / len(ep)
    packed_in = {"samples_per_s": n_sample / (packed_ms * 1e-3), "avg_launch_ms": packed_ms,
                 "bytes_per_sample": n * 1536 + 16,
                 "hbm_gbs": n_sample * (n * 1536 + 16) / (packed_ms * 1e-3) / 1e9,
                 "api": "no_trace_eval_packed (NO_PACK_CHARGE vertices, 2.0 GB per launch)"}
    del d_P
    bytes_step = n_sample * (n * 4096 + 16)
    peak, peak_src = hbm_peak_gbs()
    achieved = bytes_step * steps / (sum(step_ms) * 1e-3) / 1e9
    useful_gbs = n_sample * (n * 1536 + 16) * steps / (sum(step_ms) * 1e-3) / 1e9
    # FP64 work actually issued: 8x8x4 tensor-core products (512 flops each) of the 16x16x16 steps + the folded last
    # vertex (256 complex multiply-adds)
    flops_sample = 512.0 * info["tensor_products_per_sample"] + 8.0 * 256
    flops_step = flops_sample * n_sample

    # ---- end to end: HOST momentum configurations -> no_eval (the vertices are produced on the device, where the
    # trace consumes them: the paper's pipeline) -> no_trace_eval -> HOST traces ----
    e2e = None
    if not args.no_e2e:
        m = 1 << 15                                            # samples of the pipeline leg (5 x 2^15 configurations)
        run = workloads.workload("cfg3").runs[0].shrunk(n * m, 16)
        h_cfg = torch.from_numpy(run.configurations()).pin_memory()
        h_res = torch.empty((m,), dtype=torch.complex128).pin_memory()
        d_cfg = torch.empty((n * m, 9), dtype=torch.float64, device=dev)
        d_M = torch.empty((n * m, 16, 16, 2), dtype=torch.float64, device=dev)
        d_res = torch.empty((m,), dtype=torch.complex128, device=dev)
        h = binding.no_init(device=local, **run.params())

        def pipeline():
            d_cfg.copy_(h_cfg, non_blocking=True)
            binding.no_eval(h, d_cfg.data_ptr(), n * m, d_M.data_ptr(), stream.cuda_stream)
            binding.no_trace_eval(plan, d_M.data_ptr(), m, d_res.data_ptr(), stream.cuda_stream)
            h_res.copy_(d_res, non_blocking=True)
            torch.cuda.synchronize(dev)

        pipeline()
        barrier()
        k = 5
        t0 = time.perf_counter()
        for _ in range(k):
            pipeline()
        barrier()
        t_e2e = replicas.max_over_ranks((time.perf_counter() - t0) / k, dev)
        # share of the trace inside the pipeline, device-timed
        ea, eb = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ea.record(stream)
        binding.no_trace_eval(plan, d_M.data_ptr(), m, d_res.data_ptr(), stream.cuda_stream)
        eb.record(stream)
        torch.cuda.synchronize(dev)
        e2e = {"value": world * m / t_e2e, "unit": "samples/s", "h2d_bytes_per_step": int(h_cfg.numel() * 8),
               "d2h_bytes_per_step": int(m * 16), "ms_per_step": t_e2e * 1e3, "steps": k,
               "checksum": float(h_res.abs().sum()),
               "trace_ms_inside": ea.elapsed_time(eb),
               "api": f"host configurations -> no_eval (SNM kF=1.33, 16^3 k3 grid, {n * m} vertices) -> no_trace_eval "
                      f"({m} samples) -> host traces"}
        binding.no_free(h)

    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        from oracle import trace as T
        mcpu = args.cpu_sample or (1024 if n <= 5 else 64)
        t0 = time.perf_counter()
        T.trace_bruteforce(topo, V[:mcpu])
        dt = time.perf_counter() - t0
        cpu = {"value": mcpu / dt, "unit": "samples/s", "cores": os.cpu_count(), "kind": f"oracle (brute force over 4^{2 * n} label configurations, long double)",
               "sample": f"first {mcpu} samples of the workload ({dt:.1f} s)"}
    binding.no_trace_free(plan)
    if world > 1:
        torch.distributed.destroy_process_group()
    if rank != 0:
        return
    print(json.dumps({
        "metric": TRACE_METRIC, "value": value, "unit": "samples/s", "n_gpus": world, "steps": steps, "warmup": warmup,
        "ms_per_step": t_dev / steps * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": args.workload, "description": f"spin-isospin trace of an order-{n} ring diagram ({n} vertices, {2 * n} lines, "
                   f"4^{2 * n} label configurations per sample), {n_sample} samples of seeded charge-conserving complex 16x16 vertex matrices",
                   "n_sample": n_sample, "label_configurations_per_s": value * labels, "plan": info,
                   "l2": "256 MiB buffer rewritten between timed steps (L2 flush); the input (3-5 GB) exceeds L2",
                   "parallelism": "replicas only: every rank traces the whole batch"},
        "clocks": clocks, "e2e": e2e, "gpu_launches": steps,
        # The numerator is the USEFUL bytes: with a charge-conserving plan the method needs only the 96 allowed entries of
        # a vertex (1536 B), whichever form the caller passes.  The unpacked launch also reads the 160
        # structural zeros of every matrix; that rate is reported beside it (`hbm_gbs_all_bytes_read`), not as the fraction.
        "roofline": {"bound": "hbm", "achieved": useful_gbs, "peak": peak, "unit": "GB/s", "frac": useful_gbs / peak,
                     "limiter": "latency / shared-memory occupancy (8 warps per SM, profiles/r02b.md), not HBM: the packed input "
                                "moves 2.66x fewer bytes at the same samples/s",
                     "useful_bytes_per_sample": n * 1536 + 16,
                     "hbm_gbs_all_bytes_read": achieved, "frac_all_bytes_read": achieved / peak,
                     "traffic": NCU_DRAM_BYTES_PER_LAUNCH.get(args.workload), "traffic_source": NCU_DRAM_SOURCE.get(args.workload),
                     "peak_source": peak_src, "algorithmic_bytes_per_launch": n_sample * (n * 1536 + 16),
                     "bytes_read_per_launch": bytes_step,
                     "bytes_per_sample": n * 4096 + 16, "kernel": "trace_kernel", "avg_launch_ms": sum(step_ms) / steps,
                     "fp64_tflops": flops_step * steps / (sum(step_ms) * 1e-3) / 1e12,
                     "fp64_frac_of_nominal": flops_step * steps / (sum(step_ms) * 1e-3) / 1e12 / FP64_PEAK_NOMINAL_TFLOPS,
                     "flops_per_sample": flops_sample,
                     "dense_plan_samples_per_s": dense_rate, "packed_input": packed_in,
                     "dense_plan_flops_per_sample": 8.0 * info["cmacs_per_sample"]},
        "cpu_baseline": cpu}), flush=True)


def main():
    args = parse_args()
    if args.workload == "hf":
        run_hf(args)
        return
    if args.workload in TRACE_BENCHES:
        run_trace(args)
        return
    from paper_2603_24532_b200 import workloads
    wl = workloads.workload(args.workload)
    if args.impl == "reference":
        run_reference(args, wl)
    else:
        run_b200(args, wl)


if __name__ == "__main__":
    main()
