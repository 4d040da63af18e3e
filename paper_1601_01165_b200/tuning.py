"""Shipped tuning results (step a8): winners of dedisp_tune on a B200, one text line per
(GPU, setup), in the format dedisp_tune appends.  `python -m paper_1601_01165_b200.tuning`
re-tunes the five BASELINE.json configs and the paper's two setups (or the ones named on the command
line, keeping the other entries) on the current GPU and rewrites the file."""
from __future__ import annotations

import os
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SHIPPED = os.path.join(HERE, "tuned", "b200.tsv")


def apply_shipped(plan, nr_beams: int = 1) -> bool:
    """Select the persisted winner for this plan's setup and batch size, if the shipped file has one.
    Returns whether an entry was applied (False: the plan keeps its cost-model default)."""
    return os.path.exists(SHIPPED) and plan.load_tuning(SHIPPED, nr_beams)


def merge_entries(old_text: str, new_text: str) -> str:
    """The cache file after a (partial) retune: the old entries whose key (text before the first tab) was
    not retuned, then the new ones."""
    fresh = [l for l in new_text.splitlines() if l.strip()]
    keys = {l.split("\t")[0] for l in fresh}
    kept = [l for l in old_text.splitlines() if l.strip() and l.split("\t")[0] not in keys]
    return "\n".join(kept + fresh) + "\n"


def retune(names=None, out_path: str = SHIPPED, beams_cap: int = 8) -> None:
    import torch

    from . import dedisp, workloads as wl
    names = names or list(wl.ALL)
    tmp = out_path + ".new"
    if os.path.exists(tmp):
        os.remove(tmp)
    for name in names:
        s = wl.ALL[name]
        plan = dedisp.Plan(*s.plan_args())
        nb = min(s.nr_beams, beams_cap)
        in_dt = torch.uint8 if s.in_dtype == wl.U8 else torch.float32
        d_in = torch.zeros((nb, s.nr_channels, plan.in_pitch), dtype=in_dt, device="cuda")
        d_out = torch.empty((nb, s.nr_dms, s.nr_samples), dtype=torch.float32, device="cuda")
        plan.reserve(nb)
        ms = plan.tune(d_in, d_out, nr_beams=nb, cache_path=tmp)
        for v, t in sorted(ms.items(), key=lambda kv: kv[1]):
            print("%-10s %9.4f ms  %s" % (name, t, dedisp.variant_name(v)))
        plan.destroy()
    old = open(out_path).read() if os.path.exists(out_path) else ""
    with open(tmp) as f:
        merged = merge_entries(old, f.read())
    with open(tmp, "w") as f:
        f.write(merged)
    os.replace(tmp, out_path)


if __name__ == "__main__":
    retune(sys.argv[1:] or None)
