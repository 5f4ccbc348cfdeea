#!/usr/bin/env python
"""bench.py -- throughput of one RK3 dycore step (all acoustic substeps included) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 1..5] [--impl ours|reference]

Prints ONE JSON line (rank 0).  A "step" is one erf_rk3_step of the whole hot path over the
synthetic workload; the metric is BASELINE.json's: fp64 cell-updates per second per RK3 step.
Default workload: BASELINE config 5 (1024x1024x128, the configuration the roofline target is
quoted on).  N > 1 runs N independent replicas, one per GPU (the path does not shard in this
build: DESIGN.md "Multi-GPU"), so scaling is "weak".  `--impl reference` times the CPU oracle.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "fp64 cell-updates/sec per RK3 step (incl. acoustic substeps)"
UNIT = "cell-updates/s"
ORACLE_SAMPLE = dict(nx=64, ny=64)  # bounded sample of the workload for the CPU legs (full nz)


# ----------------------------------------------------------------------------- helpers
def algorithmic_doubles(case):
    """SURVEY.md 8(d) / DESIGN.md: compulsory fp64 words per cell for the slow RHS (per stage),
    one substep, and the three stage init/finish combines."""
    terrain = case.get("z_nodes") is not None
    slow = 12 + (2 if case["params"]["diffusion"] == 2 else 0) + (3 if terrain else 0)
    sub = 20 + (3 if terrain else 0)
    ns = case["ns"]
    nsub = 1 + ns // 2 + ns
    return dict(slow=slow, substep=sub, combine=30, nsub=nsub, total=3 * slow + nsub * sub + 30)


def measured_peak_gbs():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def measured_traffic(kernel_class, config):
    """DRAM bytes per launch of a kernel class from the committed ncu capture of config 5
    (profiles/r2_dram_traffic.csv: dram__bytes_read.sum + dram__bytes_write.sum); None for other workloads."""
    if config != 5:
        return None
    import csv
    try:
        with open(os.path.join(ROOT, "profiles", "r2_dram_traffic.csv")) as f:
            for row in csv.DictReader(f):
                if row["kernel_class"] == kernel_class:
                    return float(row["bytes_per_launch"])
    except Exception:
        pass
    return None


def max_over_ranks(ms, dist, device):
    """Step time of the whole job = the slowest rank's device time (all_reduce MAX); identity for one rank."""
    if dist is None:
        return float(ms)
    import torch
    t = torch.tensor([ms], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_value(world, cells, steps, ms):
    """Whole-job throughput: every rank advances its own replica of `cells` cells by `steps` steps in `ms`."""
    return world * cells * steps / (ms * 1e-3)


class ClockSampler:
    """Samples SM clock and throttle reasons during the timed region (pynvml)."""

    def __init__(self, index):
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self._stop = threading.Event()
        self._thr = None
        self.index = index

    def _run(self):
        try:
            import pynvml as nv
            nv.nvmlInit()
            h = nv.nvmlDeviceGetHandleByIndex(self.index)
            self.max_mhz = nv.nvmlDeviceGetMaxClockInfo(h, nv.NVML_CLOCK_SM)
            names = {getattr(nv, k): k for k in dir(nv) if k.startswith("nvmlClocksThrottleReason")}
            while not self._stop.is_set():
                self.samples.append(nv.nvmlDeviceGetClockInfo(h, nv.NVML_CLOCK_SM))
                r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(h)
                for bit, name in names.items():
                    if isinstance(bit, int) and bit and (r & bit) == bit and "None" not in name and "All" not in name:
                        self.reasons.add(name.replace("nvmlClocksThrottleReason", ""))
                time.sleep(0.05)
        except Exception as e:  # pragma: no cover
            self.reasons.add(f"sampler_error:{type(e).__name__}")

    def __enter__(self):
        self._thr = threading.Thread(target=self._run, daemon=True)
        self._thr.start()
        return self

    def __exit__(self, *a):
        self._stop.set()
        self._thr.join(timeout=2)

    def summary(self):
        s = sorted(self.samples)
        rename = {"SwPowerCap": "sw_power_cap", "HwSlowdown": "hw_slowdown", "HwThermalSlowdown": "hw_thermal_slowdown",
                  "SwThermalSlowdown": "sw_thermal_slowdown", "GpuIdle": "gpu_idle",
                  "ApplicationsClocksSetting": "applications_clocks_setting", "HwPowerBrakeSlowdown": "hw_power_brake",
                  "SyncBoost": "sync_boost", "DisplayClockSetting": "display_clock_setting"}
        return {"sm_mhz": s[len(s) // 2] if s else None, "sm_max_mhz": self.max_mhz,
                "reasons": sorted(rename.get(r, r) for r in self.reasons if r != "GpuIdle")}


def time_oracle(case_kw, config, steps, warmup):
    """The CPU oracle, as it stands, on a bounded sample (a periodic crop, full nz) of the workload."""
    from oracle import erfo
    from paper_2412_04395_b200 import workloads as wl
    erfo.build()
    case = wl.make_case(config, **case_kw)
    o = erfo.Oracle(case)
    o.set_state(*case["state"])
    for _ in range(warmup):
        o.step(case["dt"], case["ns"])
    t0 = time.perf_counter()
    for _ in range(steps):
        o.step(case["dt"], case["ns"])
    dt = time.perf_counter() - t0
    cells = case["nx"] * case["ny"] * case["nz"]
    return cells * steps / dt, dt / steps, f"{case['nx']}x{case['ny']}x{case['nz']} periodic crop of config {config}, {steps} steps"


def sample_kw(config):
    from paper_2412_04395_b200 import workloads as wl
    r = wl.CONFIGS[config]
    return dict(nx=min(ORACLE_SAMPLE["nx"], r["nx"]), ny=min(ORACLE_SAMPLE["ny"], r["ny"]))


def config_desc(case, config):
    p = case["params"]
    return {"workload": f"BASELINE config {config}: {case['nx']}x{case['ny']}x{case['nz']} cells, "
                        f"adv order {p['adv_order_h']}/{p['adv_order_v']}, diffusion {p['diffusion']}, "
                        f"{'terrain' if case.get('z_nodes') is not None else 'flat'}, dt={case['dt']}, "
                        f"{case['ns']} acoustic substeps",
            "cells": case["nx"] * case["ny"] * case["nz"], "n_acoustic": case["ns"], "dt": case["dt"]}


# ----------------------------------------------------------------------------- reference arm
def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    from paper_2412_04395_b200 import workloads as wl
    kw = sample_kw(args.config)
    value, spp, sample = time_oracle(kw, args.config, args.steps, args.warmup)
    case = wl.make_case(args.config, with_state=False, **kw)
    cfg = config_desc(case, args.config)   # the crop's own nx, ny and cell count
    full = wl.CONFIGS[args.config]
    cfg["workload"] = (f"{case['nx']}x{case['ny']}x{case['nz']} periodic crop of BASELINE config {args.config} "
                       f"(full size {full['nx']}x{full['ny']}x{full['nz']}); " + cfg["workload"].split(": ", 1)[1])
    cfg["sample_of"] = f"config {args.config}"
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": spp * 1e3, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic", "config": cfg,
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))
    return 0


def median(xs):
    xs = sorted(xs)
    return xs[len(xs) // 2]


def path_label(case):
    """Which kernels erf_rk3_step picks for this case on ERF_PATH_AUTO (mirrors the library's host-side selection, so that
    a fallback shows in the JSON line): k_slow_adv needs an even nx and nz + 1 <= 320, otherwise the round-1 slow-RHS
    kernels run."""
    if case.get("z_nodes") is not None:
        return "terrain: fused advection + general diffusion passes + fused terrain substeps"
    if case["nx"] % 2 == 0 and case["nz"] + 1 <= 320:
        return "fused flat kernels"
    return "fused flat kernels, round-1 slow RHS (k_slow_adv needs even nx and nz + 1 <= 320)"


def time_config(binding, wl, torch, config, steps, warmup, repeats, graph, device):
    """One configuration, device-resident: median over `repeats` of the CUDA-event time of `steps` steps, the state
    reset before every repeat; on a side stream so that the CUDA-graph option can capture."""
    case = wl.make_case(config)
    cells = case["nx"] * case["ny"] * case["nz"]
    dyc = binding.Dycore(case, device=device)
    if graph:
        dyc.set_option(binding.ERF_OPT_GRAPH, 1)
    dev = [torch.from_numpy(a).to(device) for a in case["state"]]
    side = torch.cuda.Stream()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    times = []
    torch.cuda.synchronize()
    with torch.cuda.stream(side):
        for rep in range(repeats):
            dyc.set_state(*dev)
            for _ in range(warmup if rep == 0 else 1):
                dyc.rk3_step(case["dt"], case["ns"])
            n0 = dyc.launch_count
            e0.record()
            for _ in range(steps):
                dyc.rk3_step(case["dt"], case["ns"])
            e1.record()
            side.synchronize()
            times.append(e0.elapsed_time(e1) / steps)
            launches = (dyc.launch_count - n0) // steps
    ms = median(times)
    ad = algorithmic_doubles(case)
    peak, _ = measured_peak_gbs()
    out = {"config": config, "grid": f"{case['nx']}x{case['ny']}x{case['nz']}", "cells": cells, "ms_per_step": ms,
           "value": cells / (ms * 1e-3), "launches_per_step": launches, "launch": "cuda_graph" if graph else "stream",
           "algorithmic_bytes_per_cell": ad["total"] * 8,
           "whole_step_frac": ad["total"] * 8 * cells / (ms * 1e-3) / 1e9 / peak,
           "path": path_label(case),
           "repeats": repeats, "steps": steps, "device_bytes": dyc.device_bytes}
    dyc.close()
    del dev
    torch.cuda.empty_cache()
    return out


# ----------------------------------------------------------------------------- our arm
def run_ours(args):
    import numpy as np
    import torch
    from paper_2412_04395_b200 import binding, workloads as wl

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback; use --impl reference for the oracle)")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    binding.load()

    case = wl.make_case(args.config)
    cells = case["nx"] * case["ny"] * case["nz"]
    dt, ns = case["dt"], case["ns"]
    dyc = binding.Dycore(case, device=f"cuda:{local}")
    if args.path:
        dyc.set_path(args.path)
    if args.variant:
        dyc.set_option(binding.ERF_OPT_VARIANT, args.variant)
    host = [torch.from_numpy(np.ascontiguousarray(a)).pin_memory() for a in case["state"]]
    dev = [h.cuda(non_blocking=True) for h in host]
    dyc.set_state(*dev)
    torch.cuda.synchronize()

    def barrier():
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(max(args.warmup, 0)):
        dyc.rk3_step(dt, ns)
    barrier()
    # ---- device-resident timing: K steps, CUDA events on the launching (current) stream, no per-kernel events
    # inside the timed region; median of `repeats` such measurements, the state reset before each
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    reps = []
    with ClockSampler(local) as clk:
        for rep in range(max(args.repeats, 1)):
            dyc.set_state(*dev)
            dyc.rk3_step(dt, ns)
            barrier()
            n0 = dyc.launch_count
            e0.record()
            for _ in range(args.steps):
                dyc.rk3_step(dt, ns)
            e1.record()
            barrier()
            reps.append(max_over_ranks(e0.elapsed_time(e1), dist, "cuda"))
            launches = dyc.launch_count - n0
    ms = median(reps)
    value = aggregate_value(world, cells, args.steps, ms)
    # ---- per-kernel-class device times: a separate pass with the library's own event brackets switched on
    dyc.set_timing(True)
    dyc.reset_timing()
    for _ in range(args.steps):
        dyc.rk3_step(dt, ns)
    barrier()
    kt = dyc.timing()
    dyc.set_timing(False)
    kt_steps = args.steps

    # ---- end to end: host buffers in, host buffers out, every step.  Every step copies its inputs from pinned host
    # memory and reads its result back; the steps are independent requests, so the copy-in of step n+1, the compute of
    # step n and the copy-out of step n-1 run on three streams over double-buffered device tensors (PCIe is full duplex).
    e2e_steps = max(1, args.steps)
    h2d = sum(h.numel() * 8 for h in host)
    d2h = h2d
    in_dev = [dev, [torch.empty_like(d) for d in dev]]
    out_dev = [dyc.empty_state(), dyc.empty_state()]
    out_host = [torch.empty_like(h).pin_memory() for h in host]  # the copies out are serialised on one stream
    s_in, s_c, s_out = torch.cuda.Stream(), torch.cuda.Stream(), torch.cuda.Stream()
    ev_in = [torch.cuda.Event() for _ in range(2)]    # inputs of buffer b are on the device
    ev_set = [torch.cuda.Event() for _ in range(2)]   # the library has copied buffer b in: it may be overwritten
    ev_c = [torch.cuda.Event() for _ in range(2)]     # result of buffer b is in out_dev[b]
    ev_out = [torch.cuda.Event() for _ in range(2)]   # out_dev[b] has been copied to the host

    def e2e_run(n):
        for it in range(n):
            b = it & 1
            with torch.cuda.stream(s_in):
                if it >= 2:
                    s_in.wait_event(ev_set[b])
                for d, h in zip(in_dev[b], host):
                    d.copy_(h, non_blocking=True)
                ev_in[b].record(s_in)
            with torch.cuda.stream(s_c):
                s_c.wait_event(ev_in[b])
                dyc.set_state(*in_dev[b])
                ev_set[b].record(s_c)
                dyc.rk3_step(dt, ns)
                if it >= 2:
                    s_c.wait_event(ev_out[b])
                dyc.get_state(out_dev[b])
                ev_c[b].record(s_c)
            with torch.cuda.stream(s_out):
                s_out.wait_event(ev_c[b])
                for h, d in zip(out_host, out_dev[b]):
                    h.copy_(d, non_blocking=True)
                ev_out[b].record(s_out)
        cur = torch.cuda.current_stream()
        for st_ in (s_in, s_c, s_out):
            cur.wait_stream(st_)

    e2e_run(2)
    barrier()
    t0 = time.perf_counter()
    e0.record()
    e2e_run(e2e_steps)
    e1.record()
    barrier()
    wall = time.perf_counter() - t0
    e2e_ms = max(e0.elapsed_time(e1), wall * 1e3)
    e2e_ms = max_over_ranks(e2e_ms, dist, "cuda")
    e2e_pipelined = aggregate_value(world, cells, e2e_steps, e2e_ms)

    # the same end to end with NO overlap: copy in, set_state, step, get_state, copy out, one after the other on one
    # stream -- what a time stepper whose next input is the previous output would see if it round-tripped every step
    def e2e_serial(n):
        for _ in range(n):
            for d, h in zip(in_dev[0], host):
                d.copy_(h, non_blocking=True)
            dyc.set_state(*in_dev[0])
            dyc.rk3_step(dt, ns)
            dyc.get_state(out_dev[0])
            for h, d in zip(out_host, out_dev[0]):
                h.copy_(d, non_blocking=True)

    e2e_serial(1)
    barrier()
    t0 = time.perf_counter()
    e0.record()
    e2e_serial(e2e_steps)
    e1.record()
    barrier()
    wall = time.perf_counter() - t0
    ser_ms = max_over_ranks(max(e0.elapsed_time(e1), wall * 1e3), dist, "cuda")
    e2e_value = aggregate_value(world, cells, e2e_steps, ser_ms)
    checksum = float(out_host[4].sum())
    assert np.isfinite(checksum), "state blew up"

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return 0

    # ---- roofline of the dominant kernel class (device events recorded inside the library)
    peak, peak_src = measured_peak_gbs()
    ad = algorithmic_doubles(case)
    dev_bytes = dyc.device_bytes
    alg_bytes = {"acoustic": ad["substep"] * 8 * cells, "slow_rhs": ad["slow"] * 8 * cells}
    dom = max(kt.items(), key=lambda kv: kv[1][1]) if kt else None
    roof = None
    if dom:
        name, (calls, tot_ms) = dom
        if name.startswith("acoustic_fused"):
            per_launch, units = alg_bytes["acoustic"], "one substep kernel"
        elif name.startswith("acoustic"):
            # the general path brackets all substeps of a stage: 1 + ns/2 + ns substeps over 3 groups per step
            per_launch, units = alg_bytes["acoustic"] * ad["nsub"] / 3.0, "all substeps of one RK stage (mean)"
        else:
            per_launch, units = alg_bytes["slow_rhs"], "one slow right-hand side"
        achieved = per_launch / (tot_ms / calls * 1e-3) / 1e9
        roof = {"bound": "hbm", "kernel": name, "achieved": achieved, "peak": peak, "unit": "GB/s",
                "frac": achieved / peak, "traffic": measured_traffic(name, args.config), "peak_source": peak_src,
                "launch_unit": units, "algorithmic_bytes_per_launch": per_launch,
                "avg_launch_ms": tot_ms / calls,
                "share_of_step": (tot_ms / kt_steps) / (ms / args.steps),
                "whole_step": {"algorithmic_bytes_per_cell": ad["total"] * 8,
                               "achieved": ad["total"] * 8 * cells * args.steps / (ms * 1e-3) / 1e9,
                               "frac": ad["total"] * 8 * cells * args.steps / (ms * 1e-3) / 1e9 / peak},
                "kernel_ms_per_step": {k: v[1] / kt_steps for k, v in kt.items()},
                "kernel_times_from": "a separate pass of the same steps with per-kernel CUDA events on"}

    if roof is not None:
        # the fp64 FMA peak of this device, measured by the library's DFMA micro-benchmark; the fp64-pipe
        # utilisation of each kernel against it is in profiles/r2_ncu_full_cfg5.md (ncu sm__pipe_fp64_cycles_active)
        try:
            roof["fp64_peak_tflops"] = binding.erf_measure_fp64_peak()
        except Exception as e:  # pragma: no cover
            roof["fp64_peak_tflops"] = None
            print(f"bench.py: fp64 peak not measured: {e}", file=sys.stderr)

    # ---- the other four BASELINE configurations (north_star: throughput on all five), a few seconds in total;
    # configs 1-2 are launch-bound: stream launches and the captured CUDA graph side by side
    all_cfg = None
    if world == 1 and args.config == 5 and not args.no_all_configs:
        dyc.close()
        del in_dev, out_dev, dev
        torch.cuda.empty_cache()
        all_cfg = []
        for cfgn, kw in ((1, dict(steps=20, warmup=5)), (2, dict(steps=10, warmup=3)), (3, dict(steps=5, warmup=3)),
                         (4, dict(steps=3, warmup=2))):
            all_cfg.append(time_config(binding, wl, torch, cfgn, repeats=5, graph=False, device=f"cuda:{local}", **kw))
            if cfgn <= 2:
                all_cfg.append(time_config(binding, wl, torch, cfgn, repeats=5, graph=True, device=f"cuda:{local}", **kw))
        all_cfg.append({"config": 5, "grid": f"{case['nx']}x{case['ny']}x{case['nz']}", "cells": cells,
                        "ms_per_step": ms / args.steps, "value": value, "launches_per_step": launches // args.steps,
                        "launch": "stream", "algorithmic_bytes_per_cell": ad["total"] * 8,
                        "whole_step_frac": roof["whole_step"]["frac"] if roof else None, "path": path_label(case),
                        "repeats": max(args.repeats, 1), "steps": args.steps})

    # ---- the oracle beside it, on a bounded sample (rank 0, N = 1 only)
    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        v, spp, sample = time_oracle(sample_kw(args.config), args.config, 3, 1)
        cpu = {"value": v, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample}

    cfg = config_desc(case, args.config)
    cfg.update({"l2": "inputs larger than L2 (every field >= 1 GB)" if cells * 8 > 256e6 else
                "fields fit in L2 (small configuration)",
                "replicas": world, "device_bytes": dev_bytes, "repeats": max(args.repeats, 1),
                "ms_per_step_repeats": [r / args.steps for r in reps],
                "path": "general" if args.path == 1 else "auto", "variant": args.variant})
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic", "config": cfg, "clocks": clk.summary(),
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                    "steps": e2e_steps, "ms_per_step": ser_ms / e2e_steps, "serial_ms_per_step": ser_ms / e2e_steps,
                    "mode": "serial: copy in, set_state, step, get_state, copy out one after the other, every step",
                    "pipelined_independent_requests": {
                        "value": e2e_pipelined, "ms_per_step": e2e_ms / e2e_steps,
                        "note": "copy-in of request n+1, compute of request n and copy-out of request n-1 on three "
                                "streams: valid for independent one-step requests, not for a time stepper"}},
            "gpu_launches": launches, "roofline": roof, "cpu_baseline": cpu, "all_configs": all_cfg}
    print(json.dumps(line))
    if all_cfg is None:
        dyc.close()
    if dist is not None:
        dist.destroy_process_group()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=5, choices=[1, 2, 3, 4, 5])
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--path", type=int, default=0, choices=[0, 1], help="0 auto (fused), 1 general kernels")
    ap.add_argument("--variant", type=int, default=0, help="ERF_VARIANT_* developer mask (include/erf_b200.h), 0 = defaults")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-all-configs", action="store_true", help="skip the configs 1-4 summary of the default run")
    ap.add_argument("--repeats", type=int, default=5, help="timed repeats of the K steps (median reported)")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
