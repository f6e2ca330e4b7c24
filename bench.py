#!/usr/bin/env python
"""bench.py -- compartment-steps/s (fp64) of the fixed-step hot path on B200.

Default workload (BASELINE.json configs[3], the one the metric's >= 50 % HBM target is quoted on):
ring-of-branching-cells, 32,768 cells x 291 compartments = 9,535,488 compartments, 33,280 NetCons,
dt = 0.025 ms (seeded synthetic stand-in for Table 1 "Ring").
`--config {1,2,3,5}` times the other BASELINE.json configs through the same code (a
bound per config -- step latency for 1, fp64 pipe for 2, HBM for 3 and 5).

One bench "step" = one cn_run advancing `dt_per_bench_step` dt of the whole model (every dt = one
pass of the whole hot path: deliver -> nrn_cur -> Hines -> update -> nrn_state -> threshold).
  value : n_node * dt-steps / device time, model resident in HBM (CUDA events, max over ranks)
  e2e   : same metric through the C ABI from HOST buffers: cn_model_create (H2D of the model) +
          cn_run + cn_get_v + cn_get_spikes (D2H) all inside the timed region
  --impl reference : the CPU oracle, as it stands, on a bounded sample of the same workload
  --traffic-from F : (no GPU) read an `ncu --page raw --csv` export and write the measured DRAM
          bytes per launch of every kernel, with the hash of the kernel sources, to
          profiles/r02_traffic.json -- the file `roofline.traffic` comes from
Multi-GPU: the path is specified for one GPU (north_star) -> replicas only; --gpus N runs N
independent replicas (no collective on the data path), scaling "weak".
"""
from __future__ import annotations

import argparse
import csv
import hashlib
import json
import os
import platform
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
METRIC = "compartment_steps_per_sec"
UNIT = "compartment-steps/s"
ORACLE_RINGS = 16          # config 4, bounded oracle sample: 16 of the 512 rings (297,984 comps)
TRAFFIC_FILE = ROOT / "profiles" / "r02_traffic.json"
# fp64 ALU peak: 148 SMs x 64 DFMA/clk x 2 flop x 1.965 GHz; a DFMA loop on the box
# reaches 36.2 TFLOP/s of it
FP64_PEAK_TFLOPS = 148 * 64 * 2 * 1.965e9 / 1e12
# fp64 operations per compartment-step as the kernels evaluate them (counted from
# cn_device.cuh: exp_lean = 34 flop, rcp_fast = 8 flop + MUFU, hh_advance = 328, HH nrn_cur = 16,
# elimination + back-substitution of a node = 22)
FLOP_HH, FLOP_NODE = 328 + 16, 22


# ---------------------------------------------------------------------------------------------
# workloads
# ---------------------------------------------------------------------------------------------

def make_workload(args):
    """-> (description, config dict, dt per bench step)."""
    import cn_workloads as W
    c = args.config
    if c == 4:
        n_types = 1024 if args.n_cell >= 32768 else max(1, args.n_cell // 32)
        desc = W.config4(n_cell=args.n_cell, n_types=n_types)
        cfg = {"workload": "config4: ring of branching cells, %d cells x 291 compartments, "
                           "1024 shape types x 32 cells shuffled, HH soma + axon-like path, pas "
                           "elsewhere, ExpSyn ring NetCons (1 ms), dt 0.025 ms" % args.n_cell,
               "l2": "state streamed per dt (~0.5 GB) exceeds the 126 MB L2; no flush needed"}
        return desc, cfg, 120
    if c == 1:
        desc = W.config1()
        cfg = {"workload": "config1: ring of 8 cells x 61 compartments, HH soma, pas dendrites, "
                           "ExpSyn ring (1 ms), IClamp on cell 0",
               "l2": "60 KB model: latency-bound, reports step latency, not a bandwidth"}
        return desc, cfg, 120
    if c == 2:
        desc = W.config2()
        cfg = {"workload": "config2: 4 rings x 64 cells x 601 compartments, HH on every "
                           "compartment, ExpSyn rings (1 ms)",
               "l2": "19 MB model: resident on chip (on-chip window mode) or in L2; fp64-bound"}
        return desc, cfg, 120
    if c == 3:
        desc = W.config3()
        cfg = {"workload": "config3: thalamocortical-shaped network, 3,560 cells / 14 types / "
                           "465,740 compartments, HH + Ca_HVA + SK + cai + pas, 1.1 M Exp2Syn, "
                           "delays 1-5 ms, Poisson IClamp drive",
               "l2": "138 MB per dt, about the size of the 126 MB L2 (mixed L2 / HBM)"}
        return desc, cfg, 120
    if c == 5:
        desc = W.config5(scale=args.scale)
        cfg = {"workload": "config5 at scale %.3g: cortex-shaped slice, %d cells x ~454 compartments "
                           "/ 55 types, 10 channel types, %d AMPA+NMDA synapses per cell, delays "
                           "0.1-10 ms" % (args.scale, len(desc["cell_first"]) - 1,
                                          len(desc["netcons"]["src"]) // (len(desc["cell_first"]) - 1)),
               "scale": args.scale,
               "l2": "state streamed per dt exceeds the 126 MB L2 at scale >= 0.05; no flush needed"}
        return desc, cfg, 40
    raise SystemExit("unknown --config")


def oracle_sample(args):
    """Bounded sample of the workload for the CPU oracle -> (description, n_dt, text)."""
    import cn_workloads as W
    c = args.config
    if c == 4:
        n_types = 1024 if args.n_cell >= 32768 else max(1, args.n_cell // 32)
        rings = ORACLE_RINGS if args.n_cell >= 64 * ORACLE_RINGS else max(1, args.n_cell // 64)
        d = W.config4(n_cell=args.n_cell, n_types=n_types, cells=list(range(rings)))
        return d, 1000, "%d of the rings of config4 (%d compartments)" % (rings, len(d["parent"]))
    if c == 1:
        d = W.config1()
        return d, 200000, "the whole of config1 (488 compartments)"
    if c == 2:
        d = W.config2(rings=[0])
        return d, 4000, "one of the four rings of config2 (%d compartments)" % len(d["parent"])
    if c == 3:
        d = W.config3()
        return d, 300, "the whole of config3 (465,740 compartments; no closed subset exists)"
    d = W.config5(n_cell=55, syn_per_cell=4000)
    return d, 200, ("a 55-cell copy of config5 with full-size cells and 4,000 synapses per cell "
                    "(%d compartments; the network has no closed subset)" % len(d["parent"]))


# ---------------------------------------------------------------------------------------------
# byte / flop models
# ---------------------------------------------------------------------------------------------

PER_INSTANCE_BYTES = {"pas": 16, "hh": 80, "expsyn": 20, "exp2syn": 36, "ampanmda": 68,
                      "iclamp": 0, "hhform": 40, "sk": 24, "cadyn": 16, "gap": 16}
POINT = ("expsyn", "exp2syn", "ampanmda", "iclamp", "gap")


def algorithmic_bytes_per_dt(desc, part="all"):
    """SURVEY.md 8(d) byte model: node 44 B (v R/W 16, a,b 16, parent 4, static diagonal 8), pas 16,
    HH 80, ExpSyn 20, Exp2Syn 36, AMPA+NMDA 68 per instance per dt; HH-form channel 40 (gbar 8,
    two gates R/W 32), SK 24, cai 16.  part: "all", "pp" (point processes) or "step" (the rest)."""
    b = 44 * len(desc["parent"]) if part in ("all", "step") else 0
    for m in desc["mechs"]:
        is_pp = m["type"] in POINT
        if part == "all" or (part == "pp") == is_pp:
            b += PER_INSTANCE_BYTES[m["type"]] * len(m["node"])
    return b


def flops_per_dt(desc):
    n_hh = sum(len(m["node"]) for m in desc["mechs"] if m["type"] == "hh")
    return FLOP_HH * n_hh + FLOP_NODE * len(desc["parent"])


def source_sha():
    """Hash of what decides the kernels' DRAM traffic: the device code and the layout / program
    compilers (not the host-side set-up and ABI code)."""
    h = hashlib.sha256()
    csrc = ROOT / "paper_1901_10975_b200" / "csrc"
    for f in sorted(list(csrc.glob("*.cuh")) + [csrc / "cn_layout.hpp", csrc / "cn_tape_program.hpp"]):
        h.update(f.name.encode())
        h.update(f.read_bytes())
    return h.hexdigest()[:16]


def write_traffic(csv_path):
    """ncu raw-page CSV -> profiles/r02_traffic.json (DRAM bytes per launch of every kernel)."""
    rows = list(csv.reader(open(csv_path, newline="")))
    hdr = next(i for i, r in enumerate(rows) if "Kernel Name" in r)
    names, units = rows[hdr], rows[hdr + 1]
    col = {n: j for j, n in enumerate(names)}
    scale = {"byte": 1, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "Tbyte": 1e12,
             "ns": 1, "us": 1e3, "ms": 1e6, "s": 1e9}

    def val(r, name):
        return float(r[col[name]].replace(",", "")) * scale[units[col[name]]]

    out = {}
    for r in rows[hdr + 2:]:
        if len(r) <= col["dram__bytes_read.sum"] or not r[col["Kernel Name"]]:
            continue
        k = r[col["Kernel Name"]].split("(")[0].replace("cn::", "").replace("void ", "").split("<")[0]
        e = out.setdefault(k, {"launches": 0, "dram_bytes": 0.0, "duration_ns": 0.0})
        e["launches"] += 1
        e["dram_bytes"] += val(r, "dram__bytes_read.sum") + val(r, "dram__bytes_write.sum")
        if "gpu__time_duration.sum" in col:
            e["duration_ns"] += val(r, "gpu__time_duration.sum")
    for e in out.values():
        e["dram_bytes_per_launch"] = e.pop("dram_bytes") / e["launches"]
        e["duration_ns_per_launch"] = e.pop("duration_ns") / e["launches"]
    prev = json.loads(TRAFFIC_FILE.read_text()) if TRAFFIC_FILE.exists() else {}
    key = Path(csv_path).stem.replace("_full", "").replace("r02_", "")   # r02_config4_full.csv -> "config4"
    prev[key] = {"source_sha": source_sha(), "from": Path(csv_path).name, "kernels": out}
    TRAFFIC_FILE.write_text(json.dumps(prev, indent=1, sort_keys=True) + "\n")
    print(json.dumps(prev[key]))


def measured_traffic(key, kernel):
    """DRAM bytes per launch from the committed ncu capture of this workload, or None when there
    is none or it was taken from other kernel sources than the ones being timed."""
    if not TRAFFIC_FILE.exists():
        return None, "no capture"
    e = json.loads(TRAFFIC_FILE.read_text()).get(key)
    if not e or kernel not in e["kernels"]:
        return None, "no capture"
    if e["source_sha"] != source_sha():
        return None, "capture is of other sources (%s)" % e["source_sha"]
    return e["kernels"][kernel]["dram_bytes_per_launch"], e["source_sha"]


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


def cpu_model():
    try:
        for ln in open("/proc/cpuinfo"):
            if ln.startswith("model name"):
                return ln.split(":", 1)[1].strip()
    except OSError:
        pass
    return platform.processor() or "unknown"


def time_oracle(desc, n_dt, warm_dt=0):
    from oracle import OracleModel
    o = OracleModel(desc)
    if warm_dt:
        o.run(warm_dt * DT, DT)
    t0 = time.perf_counter()
    o.run((warm_dt + n_dt) * DT, DT)
    return time.perf_counter() - t0


def cpu_baseline(args, n_dt_scale=1.0):
    d, n_dt, text = oracle_sample(args)
    n_dt = max(20, int(n_dt * n_dt_scale))
    el = time_oracle(d, n_dt)
    return {"value": len(d["parent"]) * n_dt / el, "unit": UNIT, "cores": 1, "kind": "oracle",
            "cpu": cpu_model(), "host_cores": os.cpu_count(),
            "sample": "%s x %d dt, %.1f s on one core" % (text, n_dt, el)}


def run_reference(args):
    """The oracle as it stands, on the host cores, bounded sample of the same workload."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import cn_workloads as W
    from oracle import OracleModel
    d, n_dt, text = oracle_sample(args)
    per_step = max(10, n_dt // 8)
    n_node = len(d["parent"])
    o = OracleModel(d)
    k = 0
    for _ in range(args.warmup):
        k += per_step
        o.run(k * DT, DT)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        k += per_step
        o.run(k * DT, DT)
    el = time.perf_counter() - t0
    value = n_node * per_step * args.steps / el
    sample = "%s, %d dt per step" % (text, per_step)
    cfg = {"workload": "config%d (BASELINE.json configs[%d]); the oracle integrates a bounded sample"
                       % (args.config, args.config - 1)}
    out = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT,
           "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
           "ms_per_step": 1e3 * el / args.steps, "higher_is_better": True, "scaling": "weak",
           "vs_baseline": None, "dtype": "f64", "data": "synthetic",
           "config": dict(cfg, sample_desc_sha256=W.desc_hash(d), dt_ms=DT),
           "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle",
                            "cpu": cpu_model(), "host_cores": os.cpu_count(), "sample": sample},
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
    ap.add_argument("--config", type=int, default=4, choices=[1, 2, 3, 4, 5],
                    help="BASELINE.json config (default 4: the headline workload)")
    ap.add_argument("--scale", type=float, default=1.0, help="config 5: fraction of the 20,000 cells "
                    "and of the 4,000 synapses per cell")
    ap.add_argument("--options", default="", help='cn_model_create_opts string, e.g. "onchip=0"')
    ap.add_argument("--n-cell", type=int, default=32768, help="debug: smaller config 4")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--traffic-from", default=None, metavar="NCU_RAW_CSV")
    args = ap.parse_args()
    if args.traffic_from:
        return write_traffic(args.traffic_from)
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

    desc, cfg, dt_per_step = make_workload(args)     # every rank: an independent replica
    n_node = len(desc["parent"])
    marsh = cn.marshal(desc)
    stream = torch.cuda.current_stream()
    opts = args.options or None

    # ---------------- device-resident timing -------------------------------------------------
    m = cn.Model(desc, marshalled=marsh, stream=stream.cuda_stream, options=opts)
    k = 0
    for _ in range(args.warmup):
        k += dt_per_step
        m.run_async(k * DT, DT)
    m.sync()
    mode = m.run_info()["mode"]
    windowed = mode != "per-step"
    launches0 = m.launch_count
    if windowed:        # every launch of the window kernel is bracketed by an event pair
        m.set_kernel_timing(1, 4096)
    sampler = ClockSampler(local_rank)
    sampler.start()
    barrier()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ev0.record(stream)
    for _ in range(args.steps):
        k += dt_per_step
        m.run_async(k * DT, DT)
    ev1.record(stream)
    barrier()
    m.sync()
    clocks = sampler.stop()
    ms = ev0.elapsed_time(ev1)
    launches = m.launch_count - launches0
    total_dt = dt_per_step * args.steps
    value, ms_max = aggregate(ms, n_node, total_dt, world, dist)
    run_info = m.run_info()

    # ---------------- kernel durations (CUDA events on the model's stream) ---------------------
    # Window modes: the event pairs of the timed region itself.  Per-step mode: the timed region
    # replays CUDA graphs, which take no event pairs; the same launches are then issued directly
    # for a few more bench steps with an event pair around every 3rd launch of each kernel class.
    kernels = {}
    if windowed:
        k_ms, k_n = m.get_kernel_timing()
        name = "cell_window_kernel" if mode == "onchip-window" else "tape_step_kernel"
        kernels[name] = {"ms_per_dt": k_ms / max(k_n, 1), "dt_sampled": k_n, "part": "all"}
    else:
        layout = m.layout_info()
        step_name = "tape_step_kernel" if layout["n_tape_group"] > 0 else "step_kernel"
        for which, name, part in (("step", step_name, "step"), ("pp", "pp_step_kernel", "pp"),
                                  ("deliver", "deliver_kernel", None)):
            m.select_timed_kernel(which)
            m.set_kernel_timing(3, 4096)
            for _ in range(max(1, min(args.steps, 3))):
                k += dt_per_step
                m.run_async(k * DT, DT)
            m.sync()
            k_ms, k_n = m.get_kernel_timing()
            if k_n:
                kernels[name] = {"ms_per_dt": k_ms / k_n, "dt_sampled": k_n, "part": part}
        m.set_kernel_timing(0, 0)
    n_spikes = len(m.get_spikes()[0])
    info = m.layout_info()
    m.destroy()

    # ---------------- roofline of the dominant kernel -------------------------------------------
    peaks_file = ROOT / "MEASURED_PEAKS.json"
    if peaks_file.exists():
        peak = float(json.loads(peaks_file.read_text())["hbm_gbs"])
        peak_src = "measured (MEASURED_PEAKS.json hbm_gbs)"
    else:
        peak, peak_src = 6650.0, "fallback (B200_PROFILING.md)"
    dom = max((kv for kv in kernels.items() if kv[1]["part"]), key=lambda kv: kv[1]["ms_per_dt"])
    dom_name, dom_k = dom
    dt_per_launch = run_info["window_steps"] if windowed else 1
    alg_all = algorithmic_bytes_per_dt(desc)
    alg_dom = algorithmic_bytes_per_dt(desc, dom_k["part"])
    traffic, traffic_src = measured_traffic("config%d" % args.config, dom_name)
    bound = {1: "latency", 2: "alu", 3: "hbm", 4: "hbm", 5: "hbm"}[args.config]
    common = {"kernel": "cn::" + dom_name, "kernel_ms_per_dt": dom_k["ms_per_dt"],
              "dt_sampled": dom_k["dt_sampled"], "dt_per_launch": dt_per_launch,
              "traffic": traffic, "traffic_source": traffic_src,
              "algorithmic_bytes_per_dt": alg_all,
              "kernels_ms_per_dt": {n: v["ms_per_dt"] for n, v in kernels.items()},
              "kernel_timing": "event pairs inside the timed region" if windowed else
                               "separate pass after the timed region, launches issued directly "
                               "(the timed region replays CUDA graphs)"}
    if bound == "hbm":
        achieved = alg_dom / (dom_k["ms_per_dt"] * 1e-3) / 1e9
        roofline = dict(common, bound="hbm", achieved=achieved, peak=peak, unit="GB/s",
                        frac=achieved / peak, peak_source=peak_src,
                        algorithmic_bytes_per_launch=alg_dom * dt_per_launch,
                        measured_dram_frac=(traffic / dt_per_launch / (dom_k["ms_per_dt"] * 1e-3) / 1e9 / peak)
                        if traffic else None,
                        whole_step={"achieved": alg_all / (1e-3 * ms_max / total_dt) / 1e9,
                                    "frac": alg_all / (1e-3 * ms_max / total_dt) / 1e9 / peak})
    elif bound == "alu":
        fl = flops_per_dt(desc)
        achieved = fl / (dom_k["ms_per_dt"] * 1e-3) / 1e12
        roofline = dict(common, bound="alu", achieved=achieved, peak=FP64_PEAK_TFLOPS,
                        unit="TFLOP/s", frac=achieved / FP64_PEAK_TFLOPS,
                        peak_source="derived: 148 SMs x 64 DFMA/clk x 2 x 1.965 GHz (DESIGN.md 6; "
                                    "a DFMA loop on the box reaches 36.2)",
                        flops_per_dt=fl, flops_per_hh_compartment=FLOP_HH + FLOP_NODE,
                        hbm_equivalent_us_per_dt=alg_all / (peak * 1e9) * 1e6)
    else:
        roofline = dict(common, bound="latency", achieved=1e3 * ms_max / total_dt, peak=None,
                        unit="us/dt (step latency)", frac=None,
                        peak_source="none: a 60 KB model is bound by the dependent chain of one "
                                    "step, not by a throughput")

    # ---------------- end to end from host buffers ---------------------------------------------
    e2e = None
    if not args.no_e2e:
        # (two repetitions, the faster one reported and both listed: the set-up runs on all host
        # cores of a shared box and a single sample varies by 2x)
        times = []
        for _ in range(2):
            barrier()
            t0 = time.perf_counter()
            m2 = cn.Model(desc, marshalled=marsh, stream=stream.cuda_stream, options=opts)
            m2.run(total_dt * DT, DT)
            v = m2.get_v()
            g, s = m2.get_spikes()
            torch.cuda.synchronize()
            el = time.perf_counter() - t0
            t = torch.tensor([el], dtype=torch.float64, device="cuda")
            if dist is not None:
                dist.all_reduce(t, op=dist.ReduceOp.MAX)
            times.append(float(t.item()))
            m2.destroy()
        el = min(times)
        e2e = {"value": world * n_node * total_dt / el, "unit": UNIT,
               "h2d_bytes_per_step": marsh[2] / args.steps,
               "d2h_bytes_per_step": (v.nbytes + g.nbytes + s.nbytes) / args.steps,
               "seconds": el, "seconds_all": times,
               "includes": "cn_model_create (validation, shape classes, H2D of the model) + "
                           "cn_run of all steps + cn_get_v + cn_get_spikes (D2H); best of 2"}

    # ---------------- CPU baseline: the oracle, bounded sample, rank 0 at N = 1 -------------------
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        cpu = cpu_baseline(args)

    if rank == 0:
        cfg.update({"n_cell": len(desc["cell_first"]) - 1, "n_compartment": n_node, "dt_ms": DT,
                    "dt_per_bench_step": dt_per_step, "mode": run_info, "replicas": world,
                    "layout": info, "spikes_in_run": n_spikes, "options": args.options,
                    "desc_sha256": W.desc_hash(desc),   # the input's hash with every result
                    "source_sha": source_sha()})
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
