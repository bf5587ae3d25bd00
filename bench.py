#!/usr/bin/env python
"""bench.py -- throughput of the hot path (one "step" = one pass of the whole simulation over one batch of
synthetic instances) on N GPUs of one node.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg1] [--impl ours|reference]

N=1 workload = BASELINE.json configs[3] (cfg3: 4,096 instances x 7,168 flows, the largest single-GPU configuration and
the one whose tables are HBM-resident); the same line carries `per_config`: one short run of each other config.
Prints ONE JSON line (rank 0).  `value` = flow-events/s with the tables already resident in HBM; `e2e` = the same
metric through the C-ABI from HOST arrays (submission calls, table build, H2D, run, D2H inside the timed region).
N>1: instances are independent, so each rank simulates its own block of instances (weak scaling, no data-path
collective); time = max over ranks.
--impl reference times the CPU oracle (oracle/, as it stands) on a bounded sample of the same workload.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)
sys.path.insert(0, os.path.join(ROOT, "tests"))

import numpy as np

METRIC = "flow_events_per_sec"
UNIT = "flow-events/s"


def shard_instances(total, rank, world):
    """Contiguous block of instance indices of rank `rank` (instances are independent: no collective)."""
    per = total // world
    extra = total % world
    lo = rank * per + min(rank, extra)
    return list(range(lo, lo + per + (1 if rank < extra else 0)))


def make_workload(name, n_gpus, per_gpu=0):
    """The named BASELINE.json config, `per_gpu` instances per GPU (0 = the config's own batch)."""
    from paper_2505_01616_b200 import workloads as W
    if name == "cfg0":
        return W.cfg0(), 1
    if name == "cfg1":
        return W.cfg1(batch=(per_gpu or 64) * n_gpus), per_gpu or 64
    if name == "cfg2":
        return W.cfg2(), 1
    if name == "cfg3":
        return W.cfg3(batch=(per_gpu or 4096) * n_gpus), per_gpu or 4096
    if name == "cfg4":
        return W.cfg4(batch=(per_gpu or 8) * n_gpus), per_gpu or 8
    # shrunken variants (the parity-test sizes), for profiling runs only
    if name == "cfg2s":
        return W.cfg2(k=8, agg_uplinks=2), 1
    if name == "cfg4s":
        return W.cfg4(batch=(per_gpu or 2) * n_gpus, n_hosts=8, gph=8, n_leaves=4, n_spines=2), per_gpu or 2
    if name == "a2a304":      # cfg4's recipe on 304 GPUs: 92,112 concurrent flows in one unit -> the grid path
        return W.cfg4(batch=1, n_hosts=38, gph=8, n_leaves=2, n_spines=4), 1
    raise SystemExit(f"unknown workload {name}")


# ---------------------------------------------------------------------------------------------- clocks
class ClockSampler:
    """Samples nvidia-smi SM clocks and throttle reasons during the timed region."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index = index
        self.rows = []
        self.proc = None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-i", str(self.index), "-lms", "100"], stdout=subprocess.PIPE,
                                         stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        for r in self.rows:
            try:
                sm.append(float(r[1])); mx.append(float(r[2]))
            except Exception:
                continue
            for name, v in zip(["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"], r[4:8]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


# ---------------------------------------------------------------------------------------------- oracle legs
def oracle_time(w, indices, mode=1):
    """Runs the CPU oracle (fast mode, single thread) over the given instances; returns (seconds in orc_run,
    flow count, collectives, summed work counters)."""
    from oracle import orc
    from util import oracle_build
    secs, flows, colls = 0.0, 0, 0
    work = {}
    for i in indices:
        sim = oracle_build(w.desc, w.instances[i], base_seed=w.base_seed)
        t0 = time.perf_counter()
        sim.run(mode=mode)
        secs += time.perf_counter() - t0
        flows += sim.num_flows
        colls += w.instances[i].n_collectives
        for k, v in sim.work_counters().items():
            work[k] = work.get(k, 0.0) + v
        sim.close()
    return secs, flows, colls, work


def oracle_prefix_time(w, workload):
    """cfg2 / cfg4 (one instance takes the oracle minutes): instance 0 run up to the simulated time by which a
    fraction q of its flows is done (orc_run_until; the time comes from the stored oracle output under
    tests/golden/, q chosen for 10-20 s of CPU work).  Returns (seconds in the run, flow-events processed, events,
    sample description, the golden file's contents)."""
    from oracle import orc
    from util import oracle_build
    g = np.load(os.path.join(ROOT, "tests", "golden", f"{workload}_inst0.npz"))
    q = {"cfg2": 0.10, "cfg4": 0.025}[workload]
    t_stop = float(np.quantile(g["t_done"], q))
    osim = oracle_build(w.desc, w.instances[0], base_seed=w.base_seed)
    t0 = time.perf_counter()
    osim.run(mode=orc.MODE_FAST, until=t_stop)
    secs = time.perf_counter() - t0
    elog = osim.event_log()
    fe = int(elog["n_completed"].sum()) + int(elog["n_activated"].sum())
    osim.close()
    sample = (f"instance 0 of {workload} up to simulated time {t_stop:.6g} s ({100 * q:g} % of its flows done: "
              f"{len(elog)} events, {fe} flow-events), oracle fast mode, 1 thread")
    return secs, fe, len(elog), sample, g


def algorithmic_bytes(work):
    """Algorithmic bytes of a run, summed over its events:
        Bytes_e = A(36 + 20h) + 12 Lambda_act + 40 c
    every active flow's state and path touched once per event, every active link's (cap_rem, n) once, retire +
    release per completion.  A, h, Lambda_act, c are counted by the oracle.  Also returned: SURVEY.md 8(d)'s
    figure, which charges the link term once per water-filling ITERATION of the one-bottleneck-per-iteration
    algorithm (12 Lambda_act R).  The parallel-round schedule does not execute those iterations, and with it the
    "fraction of peak" exceeds 1, so it is reported beside the headline, not as the headline."""
    base = 36.0 * work["sum_A"] + 20.0 * work["sum_Ah"] + 40.0 * work["completions"]
    return base + 12.0 * work["sum_Lam"], base + 12.0 * work["sum_LamR"]


# ---------------------------------------------------------------------------------------------- reference arm
def run_reference(args, rank, world):
    if rank != 0:
        return
    w, per_rank = make_workload(args.workload, 1)
    # bounded sample: a few instances per step so the whole run stays within minutes
    per_step = {"cfg0": 1, "cfg1": 4, "cfg2": 1, "cfg3": 8, "cfg4": 1}[args.workload]
    nxt = 0
    prefix = args.workload in ("cfg2", "cfg4")
    sample_txt = [f"{per_step} instances of {args.workload} per step (oracle fast mode, time inside orc_run only)"]
    def step():
        nonlocal nxt
        if prefix:   # minutes per instance: each step is the same time prefix of instance 0
            secs, fe, _ne, smp, _g = oracle_prefix_time(w, args.workload)
            sample_txt[0] = smp + ", every step"
            return secs, fe / 2.0, 0, None
        idx = [(nxt + k) % w.batch for k in range(per_step)]
        nxt = (nxt + per_step) % w.batch
        return oracle_time(w, idx)
    with PinnedCore() as pin:
        for _ in range(args.warmup):
            step()
        secs = flows = colls = 0
        for _ in range(args.steps):
            s, f, c, _w = step()
            secs += s; flows += f; colls += c
    val = 2.0 * flows / secs
    sample = sample_txt[0]
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * secs / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64+i64", "data": "synthetic",
        "config": {"workload": args.workload, "sample": sample},
        "collectives_per_sec": colls / secs,
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample,
                         "cpu_model": cpu_model(), "pinned_to_core": pin.core, "host_cores": os.cpu_count()},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }))


# ---------------------------------------------------------------------------------------------- our arm
def cpu_model():
    try:
        for line in open("/proc/cpuinfo"):
            if line.startswith("model name"):
                return line.split(":", 1)[1].strip()
    except Exception:
        pass
    return "unknown"


class PinnedCore:
    """Pins the calling process to one core while the single-threaded oracle is timed."""
    def __enter__(self):
        self.old = None
        try:
            self.old = os.sched_getaffinity(0)
            self.core = max(self.old)
            os.sched_setaffinity(0, {self.core})
        except Exception:
            self.core = None
        return self

    def __exit__(self, *exc):
        if self.old:
            try:
                os.sched_setaffinity(0, self.old)
            except Exception:
                pass


def golden_work(workload, n_inst):
    """Work counters of the FULL oracle runs of cfg2 / cfg4, stored beside the golden values by
    tests/golden/make_golden.py (which calls only oracle/): summed over instances 0..n_inst-1."""
    wk, flows = {}, 0
    for i in range(n_inst):
        path = os.path.join(ROOT, "tests", "golden", f"{workload}_inst{i}.npz")
        if not os.path.exists(path):
            return None, 0
        g = np.load(path)
        for k, v in zip(g["work_keys"].tolist(), g["work_vals"].tolist()):
            wk[k] = wk.get(k, 0.0) + v
        flows += int(g["n_flows"])
    return wk, flows


def measured_traffic(workload):
    """DRAM bytes per launch of the dominant kernel, from the metrics-only ncu capture of the full-size launch
    committed under profiles/ (profiles/r2_dram_traffic.csv; the .md beside it names the command)."""
    try:
        import csv
        for row in csv.DictReader(open(os.path.join(ROOT, "profiles", "r2_dram_traffic.csv"))):
            if row["workload"] == workload:
                return float(row["dram_bytes_read"]) + float(row["dram_bytes_write"]), row["kernel"]
    except Exception:
        pass
    return None, None


def measure(name, args, rank, world, local_rank, dist, steps, warmup, want_e2e, want_cpu):
    """One workload on this rank's share of the instances.  Returns the result dict on rank 0 (None elsewhere)."""
    import torch
    from paper_2505_01616_b200 import binding as B
    w, per_rank = make_workload(name, world, args.instances)
    mine = shard_instances(w.batch, rank, world)
    first, count = mine[0], len(mine)
    stream = torch.cuda.Stream()
    sp = stream.cuda_stream
    flush_buf = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")      # > 126 MB L2

    # ---- device-resident arm: tables built and uploaded once, each step = phs_run
    sim = B.Sim.from_workload(w, instances=(first, count), path=args.path, cta_slots=args.gang,
                              windows=not args.no_windows)
    sim.finalize(stream=sp)
    flows = sim.total_flows
    colls = sum(w.instances[i].n_collectives for i in mine)

    def barrier():
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    def one_step():
        flush_buf.zero_()                       # L2 flush between timed iterations (outside the events)
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        with torch.cuda.stream(stream):
            e0.record(stream)
            sim.run(stream=sp)
            e1.record(stream)
        e1.synchronize()
        return e0.elapsed_time(e1), sim.counters()

    for _ in range(warmup):
        one_step()
    barrier()
    sampler = ClockSampler(local_rank)
    if rank == 0:
        sampler.start()
    ms_total, kern_ms, launches = 0.0, 0.0, 0
    for _ in range(steps):
        ms, c = one_step()
        ms_total += ms
        kern_ms += c["main_kernel_ms"]
        launches += c["n_kernel_launches"]
    barrier()
    clocks = sampler.stop() if rank == 0 else None
    counters = sim.counters()
    paths = sorted({sim.path_of(i) for i in range(count)})
    sim.close()

    # ---- end-to-end arm: host arrays -> C-ABI submission -> table build -> H2D -> run -> D2H, every step
    def e2e_step():
        t0 = time.perf_counter()
        s2 = B.Sim.from_workload(w, instances=(first, count), path=args.path, cta_slots=args.gang,
                                 windows=not args.no_windows)
        s2.run(stream=sp)
        out = B.phs_get_all_completion_times(s2.h)
        dt = time.perf_counter() - t0
        c = s2.counters()
        s2.close()
        return dt, c["h2d_bytes"], out.nbytes + 40 * count
    e2e_steps = max(1, min(steps, 3)) if want_e2e else 0
    e2e_s, h2d, d2h = 0.0, 0, 0
    if e2e_steps:
        e2e_step()
        barrier()
        for _ in range(e2e_steps):
            dt, h2d, d2h = e2e_step()
            e2e_s += dt
        barrier()

    # ---- reduce over ranks: time = max, work = sum
    tot = torch.tensor([ms_total, e2e_s, kern_ms], dtype=torch.float64, device="cuda")
    work = torch.tensor([flows, colls, launches], dtype=torch.float64, device="cuda")
    if dist is not None:
        dist.all_reduce(tot, op=dist.ReduceOp.MAX)
        dist.all_reduce(work)
    ms_total, e2e_s, kern_ms = tot.tolist()
    flows_all, colls_all, launches_all = work.tolist()
    del flush_buf
    if rank != 0:
        return None

    value = 2.0 * flows_all * steps / (ms_total * 1e-3)
    e2e_value = 2.0 * flows_all * e2e_steps / e2e_s if e2e_steps else None
    iters = counters["n_events"]
    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": steps, "warmup": warmup,
        "ms_per_step": ms_total / steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64+i64", "data": "synthetic",
        "config": {"workload": name, "instances_per_gpu": count, "flows_per_gpu": flows,
                   "kernel_paths": paths, "l2": "flushed between timed steps (256 MiB write)",
                   "iterations_per_step": iters, "windows_per_step": counters["n_windows"],
                   "lookahead_windows": not args.no_windows,
                   "parallel_rounds_per_step": counters["sum_par_rounds"],
                   "max_active_flows": counters["max_active"], "max_state_slots": counters["max_slots"],
                   "cluster_size": counters["cluster_size"], "clusters_resident": counters["clusters_resident"],
                   "window_gang": counters["window_gang"]},
        "collectives_per_sec": colls_all * steps / (ms_total * 1e-3),
        "sim_iterations_per_sec": iters * world * steps / (ms_total * 1e-3),
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h),
                "steps": e2e_steps, "note": "host arrays -> phs_add_* -> phs_finalize (H2D) -> phs_run -> D2H"},
        "gpu_launches": int(launches_all),
        "clocks": clocks,
    }
    # ---- CPU baseline (oracle, bounded sample, one pinned core) and roofline, rank 0 at N=1 only
    if world == 1 and want_cpu:
        n_cpu = {"cfg0": 1, "cfg1": 64, "cfg2": 0, "cfg3": 96, "cfg4": 0}.get(name, 0)
        wk = None
        with PinnedCore() as pin:
            cpu_info = {"cores": 1, "kind": "oracle", "host_cores": os.cpu_count(), "cpu_model": cpu_model(),
                        "pinned_to_core": pin.core, "timer": "time.perf_counter around orc_run (ctypes call)"}
            if n_cpu:
                idx = list(range(min(n_cpu, w.batch)))
                secs, f_cpu, c_cpu, wk = oracle_time(w, idx)
                sample = f"instances 0..{len(idx) - 1} of {name} ({f_cpu} flows), oracle fast mode, 1 thread"
                out["cpu_baseline"] = dict(cpu_info, value=2.0 * f_cpu / secs, unit=UNIT, sample=sample, seconds=secs)
                # algorithmic bytes of ONE step = the oracle's per-event work counts, scaled to the whole batch
                scale = flows / float(f_cpu)
                counted = "counted by the oracle on the cpu_baseline sample and scaled by flows"
            elif name in ("cfg2", "cfg4"):
                # minutes per instance: the timed sample is a time prefix of instance 0 (oracle_prefix_time); the work
                # counters of the FULL oracle runs of every instance are stored beside the golden values
                secs, fe, _ne, sample, g = oracle_prefix_time(w, name)
                out["cpu_baseline"] = dict(cpu_info, value=fe / secs, unit=UNIT, sample=sample, seconds=secs,
                                           stored_full_run={"seconds": float(g["oracle_seconds"]),
                                                            "flows": int(g["n_flows"]), "events": int(g["n_events"]),
                                                            "note": "whole instance 0, timed where make_golden.py ran "
                                                                    "(another machine): context only"})
                wk, f_gold = golden_work(name, w.batch)
                if wk is not None:
                    scale = flows / float(f_gold)
                    counted = ("counted by the oracle over the whole of every instance (stored by "
                               "tests/golden/make_golden.py)")
        if wk is not None:
            alg, survey = algorithmic_bytes(wk)
            peaks = {}
            try:
                peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
            except Exception:
                pass
            peak = float(peaks.get("hbm_gbs", 6650.0))
            k_s = (kern_ms / steps) * 1e-3
            traffic, tkernel = measured_traffic(name)
            kernel = {"cta": "phs_cta_kernel", "cluster": "phs_cluster_kernel", "window": "phs_window_kernel"}
            out["roofline"] = {"bound": "hbm", "achieved": alg * scale / k_s / 1e9, "peak": peak,
                               "unit": "GB/s", "frac": alg * scale / k_s / 1e9 / peak, "traffic": traffic,
                               "traffic_source": "profiles/r2_dram_traffic.csv (ncu metrics-only capture of this "
                                                 "full-size launch)" if traffic is not None else None,
                               "peak_source": "MEASURED_PEAKS.json hbm_gbs (measured copy bandwidth)" if peaks
                               else "6650 GB/s (B200_PROFILING.md fallback)",
                               "kernel": "+".join(kernel.get(p, p) for p in paths),
                               "kernel_ms": kern_ms / steps,
                               "algorithmic_bytes_per_step": alg * scale,
                               "oracle_events_per_step": wk["events"] * scale,
                               "us_per_oracle_event": 1e6 * k_s / (wk["events"] * scale) * (count if name != "cfg2" else 1)
                               if name in ("cfg2", "cfg4") else None,
                               "formula": "sum over events of A(36+20h) + 12*Lambda_act + 40c (DESIGN.md sec 5), "
                                          + counted,
                               "survey_formula": {"bytes_per_step": survey * scale,
                                                  "achieved": survey * scale / k_s / 1e9,
                                                  "note": "SURVEY.md 8(d): link term charged once per sequential "
                                                          "water-filling iteration (12*Lambda_act*R)"},
                               "note": "state is shared-memory resident: the kernels are bound by the dependent "
                                       "chain of an event, not by HBM; `traffic` is the measured DRAM bytes per "
                                       "launch (the one-time table read and the result writes)"}
    return out


def run_ours(args, rank, world, local_rank):
    import torch
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (there is no CPU fallback)"
    torch.cuda.set_device(local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    out = measure(args.workload, args, rank, world, local_rank, dist, args.steps, args.warmup, not args.no_e2e,
                  not args.no_cpu_baseline)
    # ---- the other BASELINE.json configs, one short clock-sampled run each (N=1 only): every number of BASELINE.md
    # sec 4 gets a driver-side twin in the same JSON line
    if world == 1 and not args.no_per_config and rank == 0:
        per = {}
        for name in ("cfg0", "cfg1", "cfg2", "cfg3", "cfg4"):
            if name == args.workload:
                continue
            long_step = name == "cfg4"
            r = measure(name, args, rank, world, local_rank, None, 1 if long_step else 3, 1, not long_step,
                        not args.no_cpu_baseline)
            keep = {k: r[k] for k in ("value", "ms_per_step", "collectives_per_sec", "sim_iterations_per_sec", "steps",
                                      "warmup", "gpu_launches", "clocks")}
            keep["flow_events_per_sec"] = keep.pop("value")
            keep["config"] = {k: r["config"][k] for k in ("instances_per_gpu", "flows_per_gpu", "kernel_paths",
                                                          "iterations_per_step", "windows_per_step",
                                                          "parallel_rounds_per_step", "cluster_size",
                                                          "clusters_resident", "window_gang")}
            keep["e2e_flow_events_per_sec"] = r["e2e"]["value"]
            if "roofline" in r:
                keep["roofline"] = {k: r["roofline"][k] for k in ("frac", "achieved", "peak", "traffic", "kernel",
                                                                  "kernel_ms", "algorithmic_bytes_per_step")}
            if "cpu_baseline" in r:
                keep["cpu_baseline"] = {k: r["cpu_baseline"][k] for k in ("value", "unit", "cores", "sample")}
            per[name] = keep
        out["per_config"] = per
    if rank == 0:
        print(json.dumps(out))
    if dist is not None:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="cfg3",
                    help="BASELINE.json config: cfg0 .. cfg4 (default cfg3, the largest single-GPU configuration: "
                         "4,096 instances, 29.4 M flows, the one whose tables are HBM-resident)")
    ap.add_argument("--no-per-config", action="store_true",
                    help="skip the short runs of the other configs (per_config in the JSON line)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--path", type=int, default=0,
                    help="scheduler policy: 0 auto, 1 CTA path, 2 cluster path, 3 window path")
    ap.add_argument("--gang", type=int, default=0, help="with --path 3: smallest gang (CTAs per unit) of the window path")
    ap.add_argument("--no-e2e", action="store_true", help="skip the end-to-end arm (profiling runs)")
    ap.add_argument("--no-windows", action="store_true",
                    help="one global event per kernel loop iteration instead of the lookahead-window schedule")
    ap.add_argument("--instances", type=int, default=0,
                    help="instances per GPU (default: the config's own batch); smaller batches are for profiling")
    args = ap.parse_args()
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        run_reference(args, rank, world)
    else:
        run_ours(args, rank, world, local_rank)


if __name__ == "__main__":
    main()
