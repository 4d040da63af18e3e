#!/usr/bin/env python
"""bench.py -- dedispersion throughput on B200 (BASELINE.json metric).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config apertif] [--impl ours|reference]
                  [--only] [--variant V] [--tune] [--no-cpu-baseline]

A step is one pass of the whole hot path (dedisp_execute: staging, shifted accumulate, store; for
uint8 input also the pair repacking) over one synthetic batch of the named config.  `value` is
dedispersion GFLOP/s = B*D*C*S adds / s with inputs resident in HBM; `e2e` is the
same through dedisp_execute_host_async with pinned HOST buffers (H2D + kernels + D2H inside the timed
region).  The default run also times the other four BASELINE.json configs with the same event
protocol and reports them under `configs` (north star: real-time factor and beams in real time per
config); --only skips them.  The path does not shard (replicas only): with --gpus N
every rank runs the same workload on its own GPU, no collective on the data path, value = all ranks'
adds / max-over-ranks time.
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
INT_LANES_PER_SM = 128           # 32-bit integer adds: 64 lanes on the integer pipe + 64 (IMAD) on the FMA pipe
LDS_WORDS_PER_SM = 32            # shared memory: 128 bytes per clock and SM
FALLBACK_HBM_GBS = 6650.0        # B200_PROFILING.md fallback
FALLBACK_SM_MHZ = 1965.0
# dram__bytes_read.sum + dram__bytes_write.sum per step, from the ncu --set full captures summarised
# under profiles/ (the table names the file each number comes from; profiles/r03_traffic.md)
TRAFFIC_CSV = os.path.join(ROOT, "profiles", "r03_traffic.csv")
KERNEL_SOURCES = ("kernels.cuh", "kernel_tree.cuh", "gen_tree.py", "variant_defs.cuh", "shift_table.cu")


def kernel_sources_sha16():
    """First 16 hex digits of a SHA-256 over the kernel sources: ties an ncu capture to the code it measured."""
    import hashlib
    h = hashlib.sha256()
    base = os.path.join(ROOT, "paper_1601_01165_b200", "csrc")
    for f in KERNEL_SOURCES:
        h.update(f.encode())
        h.update(open(os.path.join(base, f), "rb").read())
    return h.hexdigest()[:16]


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            d = json.load(open(p))
            return float(d["hbm_gbs"]), float(d.get("sm_max_mhz", FALLBACK_SM_MHZ)), "measured"
        except Exception:
            pass
    return FALLBACK_HBM_GBS, FALLBACK_SM_MHZ, "fallback"


def ncu_traffic(config_name, variant_name):
    """(bytes per step, source) for the config if profiles/ holds a capture of this variant."""
    import csv
    try:
        rows = {r["config"]: r for r in csv.DictReader(open(TRAFFIC_CSV))}
        d = rows[config_name]
    except Exception:
        return None, None
    if d["variant"] != variant_name:
        return None, "profiles capture is of another variant: " + d["variant"]
    if d.get("kernel_sources_sha16") != kernel_sources_sha16():
        return None, "profiles capture predates the current kernel sources (sha %s)" % d.get("kernel_sources_sha16")
    return int(d["dram_bytes_per_step"]), d["source"]


def resident_bytes_per_beam(s, in_pitch, pair_pitch, vname):
    """Device bytes one beam keeps resident while it is dedispersed: its input rows, its output, and for
    the tree_u8 kernels the beam's share of the plan-owned pair workspace (4 bytes per pair,
    nr_channels x PAIR_PITCH pairs: 273 MB for survey8, 2.6x the input itself).  The 180 GB of a B200
    divided by this is the memory cap on beams held at once."""
    esz = 1 if s.in_dtype == wl.U8 else 4
    n = s.nr_channels * in_pitch * esz + s.nr_dms * s.nr_samples * 4
    if vname.startswith("tree_u8"):
        n += s.nr_channels * pair_pitch * 4
    return n


def compulsory_bytes(s, in_samples):
    """Input read once + output written once (north_star)."""
    esz = 1 if s.in_dtype == wl.U8 else 4
    return s.nr_beams * (s.nr_channels * in_samples * esz + s.nr_dms * s.nr_samples * 4)


def binding_roof(vname, s, sm_max_mhz, sm_count=SM_COUNT):
    """The on-chip roof that bounds the variant's kind of kernel, in T adds/s
    at the maximum SM clock: (bound, peak, note).  sm_count: the device's SM count (run_ours reads it from the
    device; 148 on a B200)."""
    clk = sm_max_mhz * 1e6
    if vname.startswith("tree_u8"):
        return ("alu", sm_count * INT_LANES_PER_SM * 2 * clk / 1e12,
                "packed 16-bit adds: %d SMs x 128 integer-add lanes (64 IADD3 + 64 IMAD) x 2 counters "
                "per 32-bit add x %.0f MHz; a pure add stream measures 115 of the 128 lanes" % (sm_count, sm_max_mhz))
    if vname.startswith("tree_"):
        return ("alu", sm_count * FP32_LANES_PER_SM * clk / 1e12,
                "fp32 adds: %d SMs x 128 lanes x %.0f MHz max SM clock" % (sm_count, sm_max_mhz))
    if vname.startswith("lds_"):
        return ("lds", sm_count * LDS_WORDS_PER_SM * clk / 1e12,
                "one shared-memory word per add: %d SMs x 32 words/clk x %.0f MHz (shared-memory "
                "wavefronts, not an ALU pipe, bind this kind: profiles/r02_ncu_lds_lofar.md)" % (sm_count, sm_max_mhz))
    return ("l2", sm_count * 10 * clk / 1e12,
            "no-reuse kernel: about 10 four-byte L2 loads per clk and SM (measured, DESIGN.md section 8)")


class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the load (B200_PROFILING.md)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        self.p = None
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(index), "--query-gpu=" + self.Q,
                                       "--format=csv,noheader,nounits", "-lms", "20"],
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
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in self.f.read().splitlines():
            parts = [x.strip() for x in line.split(",")]
            if len(parts) < 7:
                continue
            try:
                sm.append(float(parts[0]))
                mx.append(float(parts[1]))
                pw.append(float(parts[2]))
            except ValueError:
                continue
            for n, v in zip(names, parts[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        self.f.close()
        os.unlink(self.f.name)
        if sm:
            out.update(sm_mhz=float(np.median(sm)), sm_max_mhz=float(max(mx)), samples=len(sm),
                       sm_mhz_min=float(min(sm)), power_w_max=float(max(pw)))
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


def check_world(gpus: int, world: int) -> None:
    """--gpus N must agree with the launcher: the driver starts N ranks with torchrun; a bare
    `python bench.py --gpus 8` would silently measure one GPU."""
    if gpus != world:
        raise SystemExit("bench.py: --gpus %d but WORLD_SIZE=%d: launch with `python -m torch.distributed.run "
                         "--nnodes=1 --nproc-per-node %d --master-addr 127.0.0.1 bench.py --gpus %d ...`"
                         % (gpus, world, gpus, gpus))


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
                      % (len(rows), D, s.nr_channels, s.nr_samples, t)}


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


class Case:
    """One config on the device: plan, rotating synthetic buffer sets, the selected variant."""

    def __init__(self, s, rank, variant=None, tune=False):
        import torch

        from paper_1601_01165_b200 import dedisp, tuning
        self.s = s
        self.plan = plan = dedisp.Plan(*s.plan_args())
        B, C, D, S = s.nr_beams, s.nr_channels, s.nr_dms, s.nr_samples
        self.in_samples, self.pitch, self.pair_pitch = plan.in_samples, plan.in_pitch, plan.pair_pitch
        self.in_dt = torch.uint8 if s.in_dtype == wl.U8 else torch.float32
        self.out_dt = torch.int32 if s.in_dtype == wl.U8 else torch.float32
        esz = 1 if s.in_dtype == wl.U8 else 4
        # Rotating buffer sets so consecutive steps do not find their input in L2 (126 MB).
        self.set_bytes = B * (C * self.pitch * esz + D * S * 4)
        self.nbuf = max(2, min(4, int(np.ceil(400e6 / self.set_bytes)) + 1)) if self.set_bytes < 8e9 else 1
        gen = torch.Generator(device="cuda").manual_seed(s.seed + rank)
        self.ins, self.outs = [], []
        for _ in range(self.nbuf):
            if s.in_dtype == wl.U8:
                x = torch.randint(0, 256, (B, C, self.pitch), dtype=torch.uint8, device="cuda", generator=gen)
            else:
                x = torch.randn((B, C, self.pitch), dtype=torch.float32, device="cuda", generator=gen)
            self.ins.append(x)
            self.outs.append(torch.empty((B, D, S), dtype=self.out_dt, device="cuda"))
        plan.reserve(B)  # uint8: the whole batch in one launch
        # Auto-tuning (step a8) happens before and outside the timed region.
        if variant is not None:
            plan.set_variant(variant)
            self.tuned = "forced"
        elif tune:
            plan.tune(self.ins[0], self.outs[0], nr_beams=B)
            self.tuned = "dedisp_tune in this run"
        else:
            self.tuned = "shipped cache" if tuning.apply_shipped(plan, nr_beams=B) else "heuristic (no cache entry)"
        self.vname = dedisp.variant_name(plan.variant)
        # kernels launched per step: the dedispersion kernel, for uint8 tree variants also the repacking
        self.launches_per_step = 2 if self.vname.startswith("tree_u8") else 1

    def step(self, i, stream):
        self.plan.execute(self.ins[i % self.nbuf], self.outs[i % self.nbuf], nr_beams=self.s.nr_beams,
                          stream=stream)

    def close(self):
        self.plan.destroy()
        self.ins = self.outs = None


def time_device(case, steps, warmup, barrier, min_warm_s=0.0):
    """W warm-up steps (at least min_warm_s seconds of back-to-back launches), then K steps timed with
    CUDA events on the launching stream.  Returns (total ms, sorted per-step ms)."""
    import torch
    stream = torch.cuda.current_stream()
    t0 = time.perf_counter()
    i = 0
    while i < warmup or (time.perf_counter() - t0) < min_warm_s:
        case.step(i, stream)
        i += 1
        if i % 8 == 0:
            torch.cuda.synchronize()
    barrier()
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(steps + 1)]
    ev[0].record(stream)
    for k in range(steps):
        case.step(k, stream)
        ev[k + 1].record(stream)
    barrier()
    return ev[0].elapsed_time(ev[-1]), sorted(ev[k].elapsed_time(ev[k + 1]) for k in range(steps))


def report(case, world, total_ms, per, steps, hbm_gbs, sm_max_mhz, peak_kind, sm_count=SM_COUNT):
    """The per-config numbers the north star asks for."""
    s = case.s
    B, C, D, S = s.nr_beams, s.nr_channels, s.nr_dms, s.nr_samples
    ms_step = total_ms / steps
    adds = B * D * C * S
    kern_ms = float(np.mean(per))
    comp = compulsory_bytes(s, case.in_samples)
    bound, peak, note = binding_roof(case.vname, s, sm_max_mhz, sm_count)
    achieved = adds / (kern_ms * 1e-3) / 1e12
    traffic, src = ncu_traffic(s.name, case.vname)
    rt = (S / s.sample_rate) / (ms_step * 1e-3 / B)
    return {
        "workload": workload_name(s), "variant": case.vname, "tuning": case.tuned,
        "ms_per_step": ms_step, "ms_per_step_median": float(np.median(per)), "ms_per_step_min": float(per[0]),
        "value": aggregate_value(adds, world, ms_step * 1e-3), "unit": UNIT, "dtype": dtype_name(s),
        "real_time_factor": rt, "beams_in_real_time": int(np.floor(rt)),
        "beams_memory_cap": int(180e9 // resident_bytes_per_beam(s, case.pitch, case.pair_pitch, case.vname)),
        "roofline": {"bound": bound, "achieved": achieved, "peak": peak, "unit": "TFLOP/s",
                     "frac": achieved / peak, "traffic": traffic, "traffic_source": src, "note": note},
        "hbm_roofline": {"compulsory_bytes": comp, "achieved_gbs": comp / (kern_ms * 1e-3) / 1e9,
                         "peak_gbs": hbm_gbs, "peak_kind": peak_kind,
                         "frac": comp / (kern_ms * 1e-3) / 1e9 / hbm_gbs,
                         "frac_of_nominal_8TBs": comp / (kern_ms * 1e-3) / 8e12},
        "gpu_launches": steps * case.launches_per_step,
        "l2": "rotating %d input/output buffer sets (%.0f MB) > 126 MB L2"
              % (case.nbuf, case.nbuf * case.set_bytes / 1e6),
    }


def run_ours(args, s):
    import torch
    import torch.distributed as dist

    from paper_1601_01165_b200 import build

    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    check_world(args.gpus, world)
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    build.build()
    hbm_gbs, sm_max_mhz, peak_kind = measured_peaks()
    sm_count = torch.cuda.get_device_properties(local).multi_processor_count
    warmup = max(args.warmup, 3)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    case = Case(s, rank, variant=args.variant, tune=args.tune)
    B, C, D, S = s.nr_beams, s.nr_channels, s.nr_dms, s.nr_samples
    # clocks are sampled over the warm-up (at least 0.6 s of back-to-back launches) and the timed steps
    sampler = ClockSampler(local) if rank == 0 else None
    total_ms, per = time_device(case, args.steps, warmup, barrier, min_warm_s=0.6)
    clocks = sampler.stop() if sampler else None
    total_ms = max_over_ranks(total_ms, world)
    head = report(case, world, total_ms, per, args.steps, hbm_gbs, sm_max_mhz, peak_kind, sm_count)

    # ---- end to end through the host-buffer entry point (pinned host memory): every step uploads
    # its input, runs the kernels and downloads its result; consecutive steps overlap on the library's
    # three-stream pipeline (dedisp_execute_host_async), as a streaming real-time user would run it.
    plan, pitch = case.plan, case.pitch
    nslot = 3 if case.set_bytes < 4e9 else 1
    h_ins = [torch.empty((B, C, pitch), dtype=case.in_dt).pin_memory() for _ in range(nslot)]
    h_outs = [torch.empty((B, D, S), dtype=case.out_dt).pin_memory() for _ in range(nslot)]
    for h in h_ins:
        h.copy_(case.ins[0])
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
    # the same, one call at a time (H2D, kernels, D2H serialised); the first call allocates the
    # workspace and is not timed
    stream = torch.cuda.current_stream()
    plan.execute_host(h_ins[0], h_outs[0], nr_beams=B, stream=stream)
    t0 = time.perf_counter()
    for i in range(3):
        plan.execute_host(h_ins[0], h_outs[0], nr_beams=B, stream=stream)
    e2e_serial_s = (time.perf_counter() - t0) / 3
    h_in, h_out = h_ins[0], h_outs[0]
    e2e_s = max_over_ranks(e2e_s, world)
    adds = B * D * C * S
    e2e = {"value": aggregate_value(adds, world, e2e_s), "unit": UNIT,
           "h2d_bytes_per_step": h_in.numel() * h_in.element_size(),
           "d2h_bytes_per_step": h_out.numel() * h_out.element_size(),
           "ms_per_step": e2e_s * 1e3, "ms_per_step_unpipelined": e2e_serial_s * 1e3,
           "api": "dedisp_execute_host_async + dedisp_host_sync, %d pinned buffer sets" % nslot}
    del h_ins, h_outs, h_in, h_out
    case.close()
    torch.cuda.empty_cache()

    # ---- the other BASELINE.json configs, same event protocol (north star: per-config real-time
    # factor and beams in real time); fewer steps for the long ones
    others = {}
    if not args.only and args.variant is None:
        for name in wl.ALL:     # the BASELINE.json configs, then the paper's own two setups
            if name == s.name:
                continue
            o = wl.ALL[name]
            # a config that cannot run here (e.g. batch40's 11 GB on a smaller device) is reported as
            # such; the headline line is printed either way (single rank only: with replicas every
            # rank must reach the same collectives)
            try:
                c = Case(o, rank, tune=args.tune)
                ksteps = args.steps if o.nr_beams == 1 else max(3, args.steps // 4)
                # every config gets its own clock record, sampled over its own warm-up and timed steps
                smp = ClockSampler(local) if rank == 0 else None
                t_ms, p = time_device(c, ksteps, 3, barrier, min_warm_s=0.4)
                clk_o = smp.stop() if smp else None
                t_ms = max_over_ranks(t_ms, world)
                others[name] = report(c, world, t_ms, p, ksteps, hbm_gbs, sm_max_mhz, peak_kind, sm_count)
                others[name]["steps"] = ksteps
                others[name]["clocks"] = clk_o
                c.close()
            except Exception as e:  # noqa: BLE001
                if world > 1:
                    raise
                others[name] = {"workload": workload_name(o), "error": "%s: %s" % (type(e).__name__, e)}
            torch.cuda.empty_cache()

    if rank == 0:
        clk = (clocks or {}).get("sm_mhz") or sm_max_mhz
        head["roofline"]["note"] += "; frac at the observed clock (%.0f MHz): %.3f" % (
            clk, head["roofline"]["frac"] * sm_max_mhz / clk)
        line = {
            "metric": METRIC, "value": head["value"], "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": warmup, "ms_per_step": head["ms_per_step"], "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": head["dtype"], "data": "synthetic",
            "config": {"workload": head["workload"], "variant": head["variant"], "tuning": head["tuning"],
                       "l2": head["l2"],
                       "replicas": "N independent replicas, no collective" if world > 1 else "1"},
            "real_time_factor": head["real_time_factor"], "beams_in_real_time": head["beams_in_real_time"],
            "beams_memory_cap": head["beams_memory_cap"],
            "ms_per_step_median": head["ms_per_step_median"], "ms_per_step_min": head["ms_per_step_min"],
            "roofline": head["roofline"], "hbm_roofline": head["hbm_roofline"],
            "e2e": e2e, "gpu_launches": head["gpu_launches"], "clocks": clocks,
        }
        if others:
            line["configs"] = others
        if world == 1 and not args.no_cpu_baseline:
            line["cpu_baseline"] = cpu_baseline(s)
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default="apertif", choices=sorted(wl.ALL))
    ap.add_argument("--only", action="store_true", help="time the named config only")
    ap.add_argument("--variant", type=int, default=None, help="force a kernel variant index (implies --only)")
    ap.add_argument("--tune", action="store_true", help="run dedisp_tune before timing")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    s = wl.ALL[args.config]
    if args.impl == "reference":
        run_reference(args, s)
    else:
        run_ours(args, s)


if __name__ == "__main__":
    main()
