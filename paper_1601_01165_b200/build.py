"""Builds libdedisp_b200.so in-tree with nvcc for sm_100a (no JIT cache: the .so travels with the
repo snapshot).  `python -m paper_1601_01165_b200.build [--force]`."""
from __future__ import annotations

import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(CSRC, "build")
LIB = os.path.join(HERE, "libdedisp_b200.so")

NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-std=c++17", "-O3", "-lineinfo",
         "-Xcompiler", "-fPIC", "-Xcompiler", "-fvisibility=default"]

# (source, object name, extra defines)
UNITS = [
    ("shift_table.cu", "shift_table.o", []),
    ("plan.cu", "plan.o", []),
    ("tuner.cu", "tuner.o", []),
    ("host_pipe.cu", "host_pipe.o", []),
    ("variants_generic.cu", "variants_generic.o", []),
    ("variants_lds.cu", "variants_lds.o", []),
    ("variants_u8.cu", "variants_u8.o", []),
]


def _tree_variants():
    """(part, WD, WT, DT, TT, CC, NS, QMAX, MINB) rows of TREE_VARIANTS in variants_tree.cu (the input
    type column is skipped)."""
    import re
    text = open(os.path.join(CSRC, "variants_tree.cu")).read()
    rows = re.findall(r"^\s*X\((\d+),\s*\w+((?:,\s*\d+){8})\)", text, flags=re.M)
    return [tuple(int(x) for x in (a + b).split(",")) for a, b in rows]


TREE = _tree_variants()
UNITS += [("variants_tree.cu", "variants_tree%d.o" % t[0], ["-DTREE_PART=%d" % t[0]]) for t in TREE]
# (DT, TT, QMAX) of every TreeTile: gen_tree.py writes their add lattices
TREE_COMBOS = sorted({"%d,%d,%d" % (t[3], t[4], t[7]) for t in TREE})


def _sources_mtime() -> float:
    m = os.path.getmtime(os.path.join(HERE, "..", "include", "dedisp.h"))
    for f in os.listdir(CSRC):
        if f.endswith((".cu", ".cuh", ".h", ".py")):
            m = max(m, os.path.getmtime(os.path.join(CSRC, f)))
    return max(m, os.path.getmtime(os.path.abspath(__file__)))


def _compile(unit):
    src, obj, defs = unit
    cmd = [NVCC, *FLAGS, *defs, "-c", os.path.join(CSRC, src), "-o", os.path.join(OBJ, obj)]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError("nvcc failed: %s\n%s\n%s" % (" ".join(cmd), r.stdout, r.stderr))
    return obj


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= _sources_mtime():
        return LIB
    os.makedirs(OBJ, exist_ok=True)
    r = subprocess.run([sys.executable, os.path.join(CSRC, "gen_tree.py"),
                        os.path.join(OBJ, "tree_gen.cuh"), *TREE_COMBOS],
                       capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError("gen_tree.py failed:\n%s\n%s" % (r.stdout, r.stderr))
    with ThreadPoolExecutor(max_workers=min(8, os.cpu_count() or 1)) as ex:
        for obj in ex.map(_compile, UNITS):
            if verbose:
                print("compiled", obj)
    tmp = LIB + ".tmp.%d" % os.getpid()
    cmd = [NVCC, "-shared", "-o", tmp, *[os.path.join(OBJ, u[1]) for u in UNITS],
           "-gencode", "arch=compute_100a,code=sm_100a", "-lcudart"]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError("link failed: %s\n%s" % (" ".join(cmd), r.stderr))
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose=True))
