"""The paper's experiments on the current GPU, as markdown tables.

  python -m paper_1601_01165_b200.experiments [sweep] [zerodm] [histogram] [stream]

sweep     PAPER.md:105-107, Figs. 1-2: the two Table 2 setups (Apertif 1024 ch / 20 kHz / 1420 MHz / 300 MHz,
          LOFAR 32 ch / 200 kHz / 138 MHz / 6 MHz), trial DMs from 0 in steps of 0.25, 12 instances from 2 to
          4096 DMs, each auto-tuned (dedisp_tune) as in the paper; GFLOP/s, the winner, the real-time factor,
          and the speed-up over the no-reuse "generically tuned" kernel (Fig. 4).
zerodm    PAPER.md:157-169 (section 4.3): all trial DMs equal to 0, i.e. perfect data reuse.
histogram PAPER.md:151, Fig. 3: the distribution of GFLOP/s over the whole tuning space (every compiled variant).
stream    the real-time setting: a long single-beam series in pinned host memory, dedispersed
          in consecutive 1-s blocks with dedisp_stream_block_async (upload, kernels, download overlapped).

Inputs are zeros of the right shape (values do not affect timing); parity is the tests' business.
"""
from __future__ import annotations

import sys

import numpy as np

from . import dedisp, workloads as wl

PAPER_APERTIF = wl.Setup("apertif-paper", 1024, 1420.0, 300.0 / 1024, 20000.0, 20000, 0.0, 0.25, 2)
PAPER_LOFAR = wl.Setup("lofar-paper", 32, 138.0, 6.0 / 32, 200000.0, 200000, 0.0, 0.25, 2)
DM_COUNTS = [2, 4, 8, 16, 32, 64, 128, 256, 512, 1024, 2048, 4096]


def tune_once(setup):
    """plan + zero buffers + dedisp_tune -> ({variant: ms}, plan facts)."""
    import torch
    plan = dedisp.Plan(*setup.plan_args())
    in_dt = torch.uint8 if setup.in_dtype == wl.U8 else torch.float32
    d_in = torch.zeros((1, setup.nr_channels, plan.in_pitch), dtype=in_dt, device="cuda")
    d_out = torch.empty((1, setup.nr_dms, setup.nr_samples), dtype=torch.float32, device="cuda")
    ms = plan.tune(d_in, d_out)
    facts = {"max_shift": plan.max_shift, "winner": dedisp.variant_name(plan.variant)}
    plan.destroy()
    del d_in, d_out
    torch.cuda.empty_cache()
    return ms, facts


def gflops(setup, ms):
    return setup.adds_per_beam / (ms * 1e-3) / 1e9


def short(name):
    return (name.split(" DMsxsamples")[0] + "," + name.split("CTA,")[1].split(" outputs")[0]
            + (" lazy" if name.endswith(" lazy") else ""))


def sweep():
    print("| setup | DMs | max shift | GFLOP/s | ms | real-time factor | winner | generic GFLOP/s | tuned / generic |")
    print("|---|---|---|---|---|---|---|---|---|")
    for base in (PAPER_APERTIF, PAPER_LOFAR):
        for d in DM_COUNTS:
            s = wl.scaled(base, nr_dms=d)
            ms, facts = tune_once(s)
            best = min(ms.values())
            generic = ms[0]  # variant 0 = generic_f32
            print("| %s | %d | %d | %.0f | %.4f | %.0f | %s | %.0f | %.1fx |"
                  % (base.name, d, facts["max_shift"], gflops(s, best), best,
                     s.seconds_of_data / (best * 1e-3), short(facts["winner"]), gflops(s, generic),
                     generic / best), flush=True)


def zerodm():
    print("| setup | DMs | GFLOP/s, all DMs = 0 (perfect reuse) | winner | GFLOP/s, step 0.25 | winner |")
    print("|---|---|---|---|---|---|")
    for base in (PAPER_APERTIF, PAPER_LOFAR):
        for d in (256, 2048):
            z = wl.scaled(base, nr_dms=d, dm_step=0.0)
            r = wl.scaled(base, nr_dms=d)
            msz, fz = tune_once(z)
            msr, fr = tune_once(r)
            print("| %s | %d | %.0f | %s | %.0f | %s |"
                  % (base.name, d, gflops(z, min(msz.values())), short(fz["winner"]),
                     gflops(r, min(msr.values())), short(fr["winner"])), flush=True)


def histogram():
    for s in (wl.APERTIF, wl.LOFAR, wl.SURVEY8):
        ms, facts = tune_once(s)
        g = np.array(sorted(gflops(s, t) for t in ms.values()))
        print("\n%s: %d variants, GFLOP/s min %.0f / median %.0f / max %.0f (winner %s)"
              % (s.name, len(g), g[0], np.median(g), g[-1], short(facts["winner"])))
        edges = np.linspace(0, g[-1] * 1.0001, 11)
        hist, _ = np.histogram(g, bins=edges)
        for lo, hi, n in zip(edges[:-1], edges[1:], hist):
            print("  %7.0f - %7.0f GFLOP/s | %s %d" % (lo, hi, "#" * int(n), n))


def stream(nblocks: int = 12):
    import time

    import torch

    from . import tuning
    print("| setup | blocks | ms per block, end to end | seconds of data per second | MB uploaded per block "
          "(first block) | host<->device GB/s |")
    print("|---|---|---|---|---|---|")
    for s in (wl.APERTIF, wl.SURVEY8, wl.LOFAR_PAPER):
        plan = dedisp.Plan(*s.plan_args())
        tuning.apply_shipped(plan)
        S, M = s.nr_samples, plan.max_shift
        total = nblocks * S
        in_dt = torch.uint8 if s.in_dtype == wl.U8 else torch.float32
        h_series = torch.zeros((s.nr_channels, total + M), dtype=in_dt).pin_memory()
        h_out = torch.empty((s.nr_dms, total), dtype=torch.float32).pin_memory()
        for b in range(3):   # warm-up: workspaces, kernel attributes
            plan.stream_block_async(h_series, total + M, h_out, total, b * S)
        plan.host_sync()
        plan.stream_reset()
        plan.stream_block_async(h_series, total + M, h_out, total, 0)
        first = plan.stream_h2d_bytes
        plan.stream_block_async(h_series, total + M, h_out, total, S)
        later = plan.stream_h2d_bytes
        plan.host_sync()
        plan.stream_reset()
        t0 = time.perf_counter()
        for b in range(nblocks):
            plan.stream_block_async(h_series, total + M, h_out, total, b * S)
        plan.host_sync()
        dt = (time.perf_counter() - t0) / nblocks
        nbytes = later + s.nr_dms * S * 4
        print("| %s | %d | %.2f | %.0f | %.1f (%.1f) | %.1f |" % (s.name, nblocks, dt * 1e3, s.seconds_of_data / dt,
                                                                later / 1e6, first / 1e6, nbytes / dt / 1e9), flush=True)
        plan.destroy()
        del h_series, h_out


if __name__ == "__main__":
    what = sys.argv[1:] or ["sweep", "zerodm", "histogram", "stream"]
    for w in what:
        {"sweep": sweep, "zerodm": zerodm, "histogram": histogram, "stream": stream}[w]()
