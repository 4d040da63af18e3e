"""Writes tests/golden/oracle_digests.json.  Calls ONLY oracle/ and the seeded
input generators (never the CUDA path).  Run from the repo root:

    python tests/golden/make_oracle_golden.py

The digests freeze the oracle's shift tables and the tiny config's dedispersed
output so that a later change to the oracle's arithmetic cannot go unnoticed.
"""
import hashlib
import json
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

import oracle  # noqa: E402
from paper_1601_01165_b200 import workloads as wl  # noqa: E402


def main():
    out = {"_about": "written by tests/golden/make_oracle_golden.py from oracle/ only", "tables": {}}
    for s in (wl.TINY, wl.APERTIF, wl.LOFAR, wl.SURVEY8):
        t = oracle.shift_table(*s.table_args())
        out["tables"][s.name] = {
            "shape": list(t.shape), "max_shift": int(t.max()), "sum": int(t.astype(np.int64).sum()),
            "sha256": hashlib.sha256(np.ascontiguousarray(t).tobytes()).hexdigest(),
        }
    s = wl.TINY
    t = oracle.shift_table(*s.table_args())
    M = int(t.max())
    pitch = (s.nr_samples + M + 3) // 4 * 4
    x = wl.make_input(s, s.nr_samples + M, pitch, pulse_shifts=t[s.pulse[0]])
    o = oracle.dedisperse(x, t, s.nr_samples)[0]
    out["tiny_output"] = {
        "in_pitch": pitch, "argmax": [int(v) for v in np.unravel_index(np.argmax(o), o.shape)],
        "max": float(o.max()), "sum": float(o.sum()),
        "sha256_f32": hashlib.sha256(o.astype(np.float32).tobytes()).hexdigest(),
    }
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "oracle_digests.json")
    with open(path, "w") as f:
        json.dump(out, f, indent=1)
        f.write("\n")
    print("wrote", path)


if __name__ == "__main__":
    main()
