#!/usr/bin/env python
"""bench.py -- compartment-steps/s (fp64) of the fixed-step hot path on B200.

Workload (BASELINE.json configs[3], the one the metric's >= 50 % HBM target is quoted on):
ring-of-branching-cells, 32,768 cells x 291 compartments = 9,535,488 compartments, 33,280 NetCons,
dt = 0.025 ms (seeded synthetic stand-in for Table 1 "Ring").

One bench "step" = one cn_run advancing DT_PER_STEP dt of the whole model (every dt = one pass of
the whole hot path: deliver -> nrn_cur -> Hines -> update -> nrn_state -> threshold).
  value : n_node * dt-steps / device time, model resident in HBM (CUDA events, max over ranks)
  e2e   : same metric through the C ABI from HOST buffers: cn_model_create (H2D of the model) +
          cn_run + cn_get_v + cn_get_spikes (D2H) all inside the timed region
  --impl reference : the CPU oracle, as it stands, on a bounded sample of the same workload
Multi-GPU: the path is specified for one GPU (north_star) -> replicas only; --gpus N runs N
independent replicas (no collective on the data path), scaling "weak".
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
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parent
sys.path.insert(0, str(ROOT))

DT = 0.025
DT_PER_STEP = 120          # dt steps per bench step (3 ms of biological time = 3 windows of 40 dt)
METRIC = "compartment_steps_per_sec"
UNIT = "compartment-steps/s"
ORACLE_RINGS = 16          # bounded oracle sample: 16 of the 512 rings (1,024 cells, 297,984 comps)


def workload_config(n_cell):
    return {"workload": "config4: ring of branching cells, %d cells x 291 compartments, "
                        "1024 shape types x 32 cells shuffled, HH soma + axon-like path, pas "
                        "elsewhere, ExpSyn ring NetCons (1 ms), dt 0.025 ms" % n_cell,
            "n_cell": n_cell, "n_compartment": n_cell * 291, "dt_ms": DT,
            "dt_per_bench_step": DT_PER_STEP,
            "l2": "state streamed per dt (~0.5 GB) exceeds the 126 MB L2; no flush needed",
            "mode": "window: one launch of the interleaved kernel integrates up to min-delay "
                    "(40) dt, every dt streams the model from HBM (CN_TAPE_WINDOW=0: one launch "
                    "per dt)"}


def aggregate(ms_local, n_node, total_dt, world, dist=None, device="cuda"):
    """Replicas-only multi-GPU: every rank integrates its own replica of the
    workload, there is no data-path collective.  The job's time is the MAX over ranks of the
    device time, the job's throughput the units all ranks processed / that time."""
    import torch
    t = torch.tensor([ms_local], dtype=torch.float64, device=device)
    if dist is not None and world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    ms_max = float(t.item())
    return world * n_node * total_dt / (ms_max * 1e-3), ms_max


def m_window_hint(args):
    """Window mode (one launch per <= 40 dt) is what the library picks for this workload unless
    CN_TAPE_WINDOW=0; in per-step mode every 7th launch is sampled instead of every launch."""
    return os.environ.get("CN_TAPE_WINDOW", "1") != "0" and args.n_cell >= 8192


def total_dt_for_launches(args):
    return DT_PER_STEP * args.steps


def algorithmic_bytes_per_dt(desc):
    """SURVEY.md 8(d) byte model: node 44 B (v R/W 16, a,b 16, parent 4, static diagonal 8),
    pas 16, HH 80, ExpSyn 20, Exp2Syn 36, AMPA+NMDA 68 per instance per dt."""
    per = {"pas": 16, "hh": 80, "expsyn": 20, "exp2syn": 36, "ampanmda": 68, "iclamp": 0,
           "hhform": 40, "sk": 24, "cadyn": 16}
    b = 44 * len(desc["parent"])
    for m in desc["mechs"]:
        b += per[m["type"]] * len(m["node"])
    return b


class ClockSampler:
    """nvidia-smi clocks during the timed region (B200_PROFILING.md clocks line)."""

    def __init__(self, gpu_index):
        self.rows = []
        self.proc = None
        self.idx = gpu_index

    def start(self):
        q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,"
             "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
             "clocks_event_reasons.sw_power_cap")
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.idx), f"--query-gpu={q}",
                 "--format=csv,noheader,nounits", "-lms", "100"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append(line.strip())

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            f = [x.strip() for x in r.split(",")]
            if len(f) < 6:
                continue
            try:
                sm.append(float(f[0]))
                mx.append(float(f[1]))
            except ValueError:
                continue
            for nm, val in zip(names, f[2:6]):
                if val.lower().startswith("active"):
                    reasons.add(nm)
        return {"sm_mhz": statistics.median(sm) if sm else None,
                "sm_max_mhz": max(mx) if mx else None, "reasons": sorted(reasons),
                "samples": len(sm)}


def time_oracle(desc, n_dt, warm_dt=0):
    from oracle import OracleModel
    o = OracleModel(desc)
    if warm_dt:
        o.run(warm_dt * DT, DT)
    t0 = time.perf_counter()
    o.run((warm_dt + n_dt) * DT, DT)
    return time.perf_counter() - t0


def run_reference(args):
    """The oracle as it stands, on the host cores, bounded sample of the same workload."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import cn_workloads as W
    from oracle import OracleModel
    desc = W.config4(cells=list(range(ORACLE_RINGS)))
    n_node = len(desc["parent"])
    o = OracleModel(desc)
    k = 0
    for _ in range(args.warmup):
        k += DT_PER_STEP
        o.run(k * DT, DT)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        k += DT_PER_STEP
        o.run(k * DT, DT)
    el = time.perf_counter() - t0
    value = n_node * DT_PER_STEP * args.steps / el
    sample = ("%d of the 512 rings of config4 (%d cells, %d compartments), %d dt per step"
              % (ORACLE_RINGS, ORACLE_RINGS * 64, n_node, DT_PER_STEP))
    out = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT,
           "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
           "ms_per_step": 1e3 * el / args.steps, "higher_is_better": True, "scaling": "weak",
           "vs_baseline": None, "dtype": "f64", "data": "synthetic",
           "config": dict(workload_config(32768), sample_desc_sha256=W.desc_hash(desc)),
           "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle",
                            "sample": sample},
           "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0,
                   "d2h_bytes_per_step": 0},
           "gpu_launches": 0}
    print(json.dumps(out))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--n-cell", type=int, default=32768, help="debug: smaller workload")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.impl == "reference":
        return run_reference(args)

    import torch
    import cn_workloads as W
    from paper_1901_10975_b200.build import build
    build()
    import paper_1901_10975_b200 as cn

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: libcn has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    n_types = 1024 if args.n_cell >= 32768 else max(1, args.n_cell // 32)
    desc = W.config4(n_cell=args.n_cell, n_types=n_types)   # every rank: an independent replica
    n_node = len(desc["parent"])
    marsh = cn.marshal(desc)
    stream = torch.cuda.current_stream()

    # ---------------- device-resident timing -------------------------------------------------
    m = cn.Model(desc, marshalled=marsh, stream=stream.cuda_stream)
    k = 0
    for _ in range(args.warmup):
        k += DT_PER_STEP
        m.run_async(k * DT, DT)
    m.sync()
    launches0 = m.launch_count
    m.set_kernel_timing(1 if m_window_hint(args) else 7, 4096)
    sampler = ClockSampler(local_rank)
    sampler.start()
    barrier()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ev0.record(stream)
    for _ in range(args.steps):
        k += DT_PER_STEP
        m.run_async(k * DT, DT)
    ev1.record(stream)
    barrier()
    m.sync()
    clocks = sampler.stop()
    ms = ev0.elapsed_time(ev1)
    k_ms, k_n = m.get_kernel_timing()
    launches = m.launch_count - launches0
    total_dt = DT_PER_STEP * args.steps
    value, ms_max = aggregate(ms, n_node, total_dt, world, dist)
    n_spikes = len(m.get_spikes()[0])
    info = m.layout_info()
    m.destroy()

    # ---------------- roofline of the dominant kernel (cn::tape_step_kernel) -------------------
    # One launch integrates a window of up to min-delay (40) dt; every dt of it streams the whole
    # model from HBM once.  achieved = algorithmic bytes of the dt covered by the sampled launches
    # / their CUDA-event duration (the library times every launch on the model's stream).
    peaks_file = ROOT / "MEASURED_PEAKS.json"
    if peaks_file.exists():
        peak = float(json.loads(peaks_file.read_text())["hbm_gbs"])
        peak_src = "measured (MEASURED_PEAKS.json hbm_gbs)"
    else:
        peak, peak_src = 6650.0, "fallback (B200_PROFILING.md)"
    alg_bytes = algorithmic_bytes_per_dt(desc)
    kern_ms = k_ms / max(k_n, 1)          # per dt
    n_tape_launches = max(1, launches // 3) if launches < total_dt_for_launches(args) else None
    achieved = alg_bytes / (kern_ms * 1e-3) / 1e9 if k_n else None
    traffic = None
    tf = ROOT / "profiles" / "tape_step_kernel_traffic.txt"
    if tf.exists():
        try:
            traffic = json.loads(tf.read_text()).get("dram_bytes_per_dt")
        except (ValueError, OSError):
            traffic = None
    dt_per_launch = (DT_PER_STEP * args.steps / n_tape_launches) if n_tape_launches else 1.0
    roofline = {"bound": "hbm", "kernel": "cn::tape_step_kernel", "achieved": achieved,
                "peak": peak, "unit": "GB/s", "frac": (achieved / peak) if achieved else None,
                "traffic": traffic * dt_per_launch if traffic else None, "peak_source": peak_src,
                "algorithmic_bytes_per_launch": alg_bytes * dt_per_launch,
                "algorithmic_bytes_per_dt": alg_bytes, "dt_per_launch": dt_per_launch,
                "kernel_ms_per_dt": kern_ms, "dt_sampled": k_n}

    # ---------------- end to end from host buffers ---------------------------------------------
    e2e = None
    if not args.no_e2e:
        barrier()
        t0 = time.perf_counter()
        m2 = cn.Model(desc, marshalled=marsh, stream=stream.cuda_stream)
        m2.run(total_dt * DT, DT)
        v = m2.get_v()
        g, s = m2.get_spikes()
        torch.cuda.synchronize()
        el = time.perf_counter() - t0
        t = torch.tensor([el], dtype=torch.float64, device="cuda")
        if dist is not None:
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
        el = float(t.item())
        e2e = {"value": world * n_node * total_dt / el, "unit": UNIT,
               "h2d_bytes_per_step": marsh[2] / args.steps,
               "d2h_bytes_per_step": (v.nbytes + g.nbytes + s.nbytes) / args.steps,
               "seconds": el,
               "includes": "cn_model_create (validation, shape classes, H2D of the model) + "
                           "cn_run of all steps + cn_get_v + cn_get_spikes (D2H)"}
        m2.destroy()

    # ---------------- CPU baseline: the oracle, bounded sample, rank 0 at N = 1 -------------------
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        rings = ORACLE_RINGS if args.n_cell >= 64 * ORACLE_RINGS else max(1, args.n_cell // 64)
        sub = W.config4(n_cell=args.n_cell, n_types=n_types, cells=list(range(rings)))
        n_dt = 1000
        el = time_oracle(sub, n_dt)
        cpu = {"value": len(sub["parent"]) * n_dt / el, "unit": UNIT, "cores": 1,
               "kind": "oracle",
               "sample": "%d rings of the same workload (%d compartments) x %d dt, %.1f s"
                         % (rings, len(sub["parent"]), n_dt, el)}

    if rank == 0:
        cfg = workload_config(args.n_cell)
        cfg.update({"replicas": world, "layout": info, "spikes_in_run": n_spikes,
                    "desc_sha256": W.desc_hash(desc)})   # the input's hash with every result
        out = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world,
               "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_max / args.steps,
               "us_per_dt": 1e3 * ms_max / total_dt,
               "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
               "data": "synthetic", "config": cfg, "clocks": clocks, "e2e": e2e,
               "gpu_launches": launches, "roofline": roofline, "cpu_baseline": cpu}
        print(json.dumps(out))
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
