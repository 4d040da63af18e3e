#!/usr/bin/env python
"""bench.py -- dedispersion throughput on B200 (BASELINE.json metric).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config apertif] [--impl ours|reference]

A step is one pass of the whole hot path (dedisp_execute: staging, shifted accumulate, store) over
one synthetic batch of the named config.  `value` is dedispersion GFLOP/s = B*D*C*S adds / s
 with inputs resident in HBM; `e2e` is the same through dedisp_execute_host with
pinned HOST buffers (H2D + kernel + D2H inside the timed region).  The path does not shard
(replicas only): with --gpus N every rank runs the same workload on its own GPU,
no collective on the data path, value = all ranks' adds / max-over-ranks time.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from paper_1601_01165_b200 import workloads as wl  # noqa: E402

METRIC = "dedispersion GFLOP/s"
UNIT = "GFLOP/s"
SM_COUNT = 148
FP32_LANES_PER_SM = 128          # fp32 add issue: 4 SMSPs x 32 lanes per clock
FALLBACK_HBM_GBS = 6650.0        # B200_PROFILING.md fallback
FALLBACK_SM_MHZ = 1965.0
# dram__bytes_read.sum + dram__bytes_write.sum per launch from the ncu --set full capture of the
# same command (profiles/README.md says which file); None until captured for that config.
NCU_TRAFFIC_BYTES = {
    # profiles/r01_ncu_tree_apertif.md: 114.9 MB read + 123.9 MB written per launch
    "apertif": 114913536 + 123922432,
}


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            d = json.load(open(p))
            return float(d["hbm_gbs"]), float(d.get("sm_max_mhz", FALLBACK_SM_MHZ)), "measured"
        except Exception:
            pass
    return FALLBACK_HBM_GBS, FALLBACK_SM_MHZ, "fallback"


def compulsory_bytes(s, in_samples):
    """Input read once + output written once (north_star)."""
    esz = 1 if s.in_dtype == wl.U8 else 4
    return s.nr_beams * (s.nr_channels * in_samples * esz + s.nr_dms * s.nr_samples * 4)


class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        self.p = None
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(index), "--query-gpu=" + self.Q,
                                       "--format=csv,noheader,nounits", "-lms", "50"],
                                      stdout=self.f, stderr=subprocess.DEVNULL)
        except OSError:
            pass

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.p is None:
            return out
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.p.kill()
        self.f.flush()
        self.f.seek(0)
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in self.f.read().splitlines():
            parts = [x.strip() for x in line.split(",")]
            if len(parts) < 7:
                continue
            try:
                sm.append(float(parts[0]))
                mx.append(float(parts[1]))
            except ValueError:
                continue
            for n, v in zip(names, parts[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        self.f.close()
        os.unlink(self.f.name)
        if sm:
            out.update(sm_mhz=float(np.median(sm)), sm_max_mhz=float(max(mx)), samples=len(sm))
        out["reasons"] = sorted(reasons)
        return out


def max_over_ranks(x: float, world: int, device="cuda") -> float:
    """Replicas only: the one cross-rank step is taking the slowest rank's time."""
    if world <= 1:
        return float(x)
    import torch
    import torch.distributed as dist
    t = torch.tensor([x], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_value(adds_per_rank: int, world: int, seconds_max: float) -> float:
    """Whole-job GFLOP/s: every rank processed the same number of adds (weak scaling)."""
    return world * adds_per_rank / seconds_max / 1e9


def cpu_baseline(s, target_s: float = 12.0):
    """The oracle as it stands, on this box's host cores, on a bounded sample of the workload: a
    subset of DM rows at full C and S (each output is still the full channel sum)."""
    import oracle
    table = oracle.shift_table(*s.table_args())
    M = int(table.max())
    one = wl.scaled(s, nr_beams=1)
    x = wl.make_input(one, s.nr_samples + M, s.nr_samples + M,
                      pulse_shifts=table[s.pulse[0]] if s.pulse else None)
    threads = oracle.num_threads()

    def run(rows):
        t0 = time.perf_counter()
        oracle.dedisperse(x, table[rows], s.nr_samples)
        return time.perf_counter() - t0

    D = s.nr_dms
    probe = np.unique(np.linspace(0, D - 1, min(D, 2 * threads)).astype(int))
    t = run(probe)
    per_row = t / len(probe)
    n = int(min(D, max(len(probe), target_s / max(per_row, 1e-9))))
    rows = np.unique(np.linspace(0, D - 1, n).astype(int))
    t = run(rows)
    adds = len(rows) * s.nr_channels * s.nr_samples
    return {"value": adds / t / 1e9, "unit": UNIT, "cores": threads, "kind": "oracle",
            "sample": "%d of %d DM rows (evenly spaced) x %d channels x %d samples, 1 beam, %.1f s"
                      % (len(rows), D, s.nr_channels, s.nr_samples, t)}, (x, table)


def run_reference(args, s):
    """--impl reference: for this tier the reference arm is the CPU oracle (no reference code
    exists).  Each step is a bounded sample of the workload; rank 0 only."""
    import oracle
    if int(os.environ.get("RANK", "0")) != 0:
        return
    table = oracle.shift_table(*s.table_args())
    M = int(table.max())
    one = wl.scaled(s, nr_beams=1)
    x = wl.make_input(one, s.nr_samples + M, s.nr_samples + M,
                      pulse_shifts=table[s.pulse[0]] if s.pulse else None)
    threads = oracle.num_threads()
    D = s.nr_dms
    # size one step at about 4 s of CPU work
    probe = np.unique(np.linspace(0, D - 1, min(D, threads)).astype(int))
    t0 = time.perf_counter()
    oracle.dedisperse(x, table[probe], s.nr_samples)
    per_row = (time.perf_counter() - t0) / len(probe)
    n = int(min(D, max(threads, 4.0 / max(per_row, 1e-9))))
    rows = np.unique(np.linspace(0, D - 1, n).astype(int))
    sub = np.ascontiguousarray(table[rows])
    for _ in range(args.warmup):
        oracle.dedisperse(x, sub, s.nr_samples)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        oracle.dedisperse(x, sub, s.nr_samples)
    dt = (time.perf_counter() - t0) / args.steps
    adds = len(rows) * s.nr_channels * s.nr_samples
    val = adds / dt / 1e9
    sample = ("%d of %d DM rows (evenly spaced) x %d channels x %d samples per step, 1 beam"
              % (len(rows), D, s.nr_channels, s.nr_samples))
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt * 1e3,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": dtype_name(s),
        "data": "synthetic", "config": {"workload": workload_name(s), "sample": sample},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": threads, "kind": "oracle",
                         "sample": sample},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


def dtype_name(s):
    return "u8->u32" if s.in_dtype == wl.U8 else "f32"


def workload_name(s):
    return ("%s: %d beams x %d channels x %d DMs x %d samples, f_low %g MHz, bw %.6g MHz, %g Hz, "
            "DM step %g" % (s.name, s.nr_beams, s.nr_channels, s.nr_dms, s.nr_samples, s.f_low_MHz,
                            s.channel_bw_MHz, s.sample_rate, s.dm_step))


def run_ours(args, s):
    import torch
    import torch.distributed as dist

    from paper_1601_01165_b200 import build, dedisp, tuning

    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    build.build()
    hbm_gbs, sm_max_mhz, peak_kind = measured_peaks()

    plan = dedisp.Plan(*s.plan_args())
    in_samples, pitch = plan.in_samples, plan.in_pitch
    B, C, D, S = s.nr_beams, s.nr_channels, s.nr_dms, s.nr_samples
    in_dt = torch.uint8 if s.in_dtype == wl.U8 else torch.float32
    out_dt = torch.int32 if s.in_dtype == wl.U8 else torch.float32
    # Rotating buffer sets so consecutive steps do not find their input in L2 (126 MB).
    esz = 1 if s.in_dtype == wl.U8 else 4
    set_bytes = B * (C * pitch * esz + D * S * 4)
    nbuf = max(2, min(4, int(np.ceil(400e6 / set_bytes)) + 1)) if set_bytes < 8e9 else 1
    gen = torch.Generator(device="cuda").manual_seed(s.seed + rank)
    ins, outs = [], []
    for _ in range(nbuf):
        if s.in_dtype == wl.U8:
            x = torch.randint(0, 256, (B, C, pitch), dtype=torch.uint8, device="cuda", generator=gen)
        else:
            x = torch.randn((B, C, pitch), dtype=torch.float32, device="cuda", generator=gen)
        ins.append(x)
        outs.append(torch.empty((B, D, S), dtype=out_dt, device="cuda"))

    # Auto-tuning (step a8) happens before and outside the timed region.
    tuned = "heuristic"
    if args.variant is not None:
        plan.set_variant(args.variant)
        tuned = "forced"
    elif args.tune:
        plan.tune(ins[0], outs[0], nr_beams=B)
        tuned = "dedisp_tune in this run"
    else:
        before = plan.variant
        tuning.apply_shipped(plan)
        tuned = "shipped cache" if (os.path.exists(tuning.SHIPPED)) else "heuristic"
        del before
    vname = dedisp.variant_name(plan.variant)

    stream = torch.cuda.current_stream()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for i in range(max(args.warmup, 3)):
        plan.execute(ins[i % nbuf], outs[i % nbuf], nr_beams=B, stream=stream)
    barrier()
    sampler = ClockSampler(local) if rank == 0 else None
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps + 1)]
    barrier()
    ev[0].record(stream)
    for i in range(args.steps):
        plan.execute(ins[i % nbuf], outs[i % nbuf], nr_beams=B, stream=stream)
        ev[i + 1].record(stream)
    barrier()
    total_ms = ev[0].elapsed_time(ev[-1])
    per = sorted(ev[i].elapsed_time(ev[i + 1]) for i in range(args.steps))
    clocks = sampler.stop() if sampler else None
    total_ms = max_over_ranks(total_ms, world)
    ms_step = total_ms / args.steps

    # ---- end to end through the host-buffer entry point (pinned host memory): every step uploads
    # its input, runs the kernels and downloads its result; consecutive steps overlap on the library's
    # three-stream pipeline (dedisp_execute_host_async), as a streaming real-time user would run it.
    nslot = 3 if set_bytes < 4e9 else 1
    h_ins = [torch.empty((B, C, pitch), dtype=in_dt).pin_memory() for _ in range(nslot)]
    h_outs = [torch.empty((B, D, S), dtype=out_dt).pin_memory() for _ in range(nslot)]
    for h in h_ins:
        h.copy_(ins[0])
    e2e_steps = max(3, min(args.steps, 12))
    for i in range(3):
        plan.execute_host_async(h_ins[i % nslot], h_outs[i % nslot], nr_beams=B)
    plan.host_sync()
    barrier()
    t0 = time.perf_counter()
    for i in range(e2e_steps):
        plan.execute_host_async(h_ins[i % nslot], h_outs[i % nslot], nr_beams=B)
    plan.host_sync()
    e2e_s = (time.perf_counter() - t0) / e2e_steps
    # the same, one call at a time (H2D, kernels, D2H serialised)
    t0 = time.perf_counter()
    for i in range(2):
        plan.execute_host(h_ins[0], h_outs[0], nr_beams=B, stream=stream)
    e2e_serial_s = (time.perf_counter() - t0) / 2
    h_in, h_out = h_ins[0], h_outs[0]
    e2e_s = max_over_ranks(e2e_s, world)

    adds = B * D * C * S
    value = aggregate_value(adds, world, ms_step * 1e-3)
    secs = S / s.sample_rate
    rt = secs / (ms_step * 1e-3 / B)
    if rank == 0:
        kern_ms = float(np.mean(per))
        comp = compulsory_bytes(s, in_samples)
        clk = (clocks or {}).get("sm_mhz") or sm_max_mhz
        alu_peak = SM_COUNT * FP32_LANES_PER_SM * sm_max_mhz * 1e6 / 1e12  # T adds/s at max clock
        achieved = adds / (kern_ms * 1e-3) / 1e12
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": ms_step, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": dtype_name(s), "data": "synthetic",
            "config": {"workload": workload_name(s), "variant": vname, "tuning": tuned,
                       "l2": "rotating %d input/output buffer sets (%.0f MB) > 126 MB L2"
                             % (nbuf, nbuf * set_bytes / 1e6),
                       "replicas": "N independent replicas, no collective" if world > 1 else "1"},
            "real_time_factor": rt, "beams_in_real_time": int(np.floor(rt)),
            "beams_memory_cap": int(180e9 // (set_bytes / B)),
            "ms_per_step_median": float(np.median(per)), "ms_per_step_min": float(per[0]),
            "roofline": {"bound": "alu", "achieved": achieved, "peak": alu_peak, "unit": "TFLOP/s",
                         "frac": achieved / alu_peak,
                         "traffic": NCU_TRAFFIC_BYTES.get(s.name),
                         "note": "fp32/u32 adds per second vs 148 SMs x 128 lanes x %.0f MHz max SM "
                                 "clock; frac at the observed clock (%.0f MHz): %.3f"
                                 % (sm_max_mhz, clk, achieved / (SM_COUNT * FP32_LANES_PER_SM * clk * 1e6 / 1e12))},
            "hbm_roofline": {"compulsory_bytes": comp, "achieved_gbs": comp / (kern_ms * 1e-3) / 1e9,
                             "peak_gbs": hbm_gbs, "peak_kind": peak_kind,
                             "frac": comp / (kern_ms * 1e-3) / 1e9 / hbm_gbs,
                             "frac_of_nominal_8TBs": comp / (kern_ms * 1e-3) / 8e12},
            "e2e": {"value": aggregate_value(adds, world, e2e_s), "unit": UNIT,
                    "h2d_bytes_per_step": h_in.numel() * h_in.element_size(),
                    "d2h_bytes_per_step": h_out.numel() * h_out.element_size(),
                    "ms_per_step": e2e_s * 1e3, "ms_per_step_unpipelined": e2e_serial_s * 1e3,
                    "api": "dedisp_execute_host_async + dedisp_host_sync, %d pinned buffer sets" % nslot},
            "gpu_launches": args.steps * ((B + 65534) // 65535),
            "clocks": clocks,
        }
        if world == 1 and not args.no_cpu_baseline:
            line["cpu_baseline"], _ = cpu_baseline(s)
        print(json.dumps(line))
    plan.destroy()
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default="apertif", choices=sorted(wl.CONFIGS))
    ap.add_argument("--variant", type=int, default=None, help="force a kernel variant index")
    ap.add_argument("--tune", action="store_true", help="run dedisp_tune before timing")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    s = wl.CONFIGS[args.config]
    if args.impl == "reference":
        run_reference(args, s)
    else:
        run_ours(args, s)


if __name__ == "__main__":
    main()
