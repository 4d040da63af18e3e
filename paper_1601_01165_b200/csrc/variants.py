"""variants.py -- THE list of compiled kernel variants (step a8, "try all meaningful
combinations"): the tuning space dedisp_tune sweeps.  Adding a point is one line here; build.py
generates one translation unit per entry, the lattices gen_tree.py must emit, and the registry table
plan.cu includes (build/registry_gen.inc).  The paper generates its kernel source per parameter set at
run time; here the same parameters select template instantiations at build time.

Parameters (the paper's five, re-cast for B200):
  WD x WT   warps per CTA over DMs x time       (work-items per work-group in DM / in time)
  DT x TT   outputs per thread, DMs x samples    (elements per work-item in DM / in time)
  CC, NS    channels per pipeline stage, stages  (local-memory staging depth)
  QMAX      tree kernels: largest per-DM-step shift increment class the lattice covers
  MINB      __launch_bounds__ minimum CTAs per SM
Registers per thread ~ DT*TT + window + 16 decide the resident warps: <= 128 for 16 warps/SM, <= 168 for
12, <= 255 for 8.  TT/4 odd keeps the LDS.128 window loads bank-conflict free.
"""

# variants 0 and 1: the no-reuse "generically tuned" kernel
GENERIC = ["float", "uint8_t"]

# KIND_LDS: staged tile, one shared-memory word per add.  (In, WD, WT, DT, TT, CC, NS, MINB)
LDS = [
    ("float", 4, 2, 4, 4, 8, 3, 2),     # 16 x 256
    ("float", 8, 1, 4, 8, 8, 3, 2),     # 32 x 256
    ("float", 4, 2, 8, 4, 8, 3, 2),     # 32 x 256
    ("float", 4, 2, 4, 8, 8, 2, 2),     # 16 x 512
    ("float", 2, 4, 4, 8, 8, 2, 2),     # 8 x 1024
    ("float", 2, 4, 8, 4, 16, 2, 2),    # 16 x 512, deeper chunk
    ("float", 2, 2, 2, 2, 8, 2, 4),     # 4 x 128 (small problems)
    ("float", 1, 8, 8, 4, 16, 2, 2),    # 8 x 1024
    ("float", 2, 4, 8, 8, 16, 2, 1),    # 16 x 1024
    # more adds per shift load and per staged byte (LOFAR-like: shared-memory wavefronts bind)
    ("float", 4, 2, 4, 16, 8, 2, 2),    # 16 x 1024
    ("float", 4, 2, 8, 8, 8, 2, 2),     # 32 x 512
    ("float", 4, 2, 8, 16, 8, 2, 1),    # 32 x 1024
    ("float", 2, 4, 8, 16, 8, 2, 1),    # 16 x 2048
    ("float", 4, 4, 4, 16, 8, 2, 1),    # 16 x 2048, 16 warps
    # long shifts (the paper's LOFAR setup, DM step 0.25: up to ~900 samples per DM step): few channels
    # per stage so that the long spans of a DM tile still fit shared memory
    ("float", 1, 8, 4, 8, 2, 3, 1),     # 4 x 2048, cc2
    ("float", 1, 8, 4, 16, 2, 3, 1),    # 4 x 4096, cc2
    ("float", 1, 8, 4, 16, 4, 2, 1),    # 4 x 4096, cc4
    ("uint8_t", 4, 2, 4, 4, 16, 3, 2),  # 16 x 256
    ("uint8_t", 8, 1, 4, 8, 16, 3, 2),  # 32 x 256
    ("uint8_t", 4, 2, 8, 4, 16, 3, 2),  # 32 x 256
    ("uint8_t", 4, 2, 8, 8, 16, 2, 2),  # 32 x 512
    ("uint8_t", 2, 2, 2, 2, 8, 2, 4),   # 4 x 128
]

# KIND_TREE: register window + generated branch lattice.  (In, WD, WT, DT, TT, CC, NS, QMAX, MINB)
# fp32: TT samples per thread and DM.  uint8: TT PAIRS of samples per thread and DM (2*TT outputs).
TREE = [
    # ---- fp32, 12 warps/SM (<= 168 registers)
    ("float", 12, 1, 4, 28, 16, 3, 3, 1),   # 48 x 896: the round-1 Apertif winner
    ("float", 12, 1, 4, 28, 8, 4, 3, 1),
    ("float", 12, 1, 4, 28, 12, 4, 3, 1),
    ("float", 12, 1, 4, 20, 8, 4, 4, 1),    # 48 x 640, q <= 4
    ("float", 12, 1, 4, 20, 16, 3, 4, 1),
    ("float", 12, 1, 5, 20, 8, 4, 3, 1),    # 60 x 640
    ("float", 12, 1, 5, 20, 16, 3, 3, 1),
    ("float", 12, 1, 8, 12, 8, 4, 4, 1),    # 96 x 384
    ("float", 12, 1, 6, 12, 16, 3, 4, 1),   # 72 x 384
    # ---- fp32, 16 warps/SM (<= 128 registers)
    ("float", 16, 1, 6, 12, 8, 4, 4, 1),    # 96 x 384
    ("float", 16, 1, 6, 12, 16, 3, 4, 1),
    ("float", 16, 1, 4, 12, 16, 3, 4, 1),   # 64 x 384
    ("float", 16, 1, 5, 12, 16, 3, 3, 1),   # 80 x 384
    ("float", 16, 1, 4, 20, 16, 3, 3, 1),   # 64 x 640
    ("float", 16, 1, 4, 20, 12, 4, 3, 1),
    ("float", 16, 1, 4, 20, 20, 3, 3, 1),
    ("float", 16, 1, 4, 20, 8, 4, 3, 1),
    # ---- fp32, 8 warps/SM (<= 255 registers)
    ("float", 8, 1, 8, 20, 8, 4, 3, 1),     # 64 x 640
    ("float", 8, 1, 8, 20, 8, 4, 4, 1),
    ("float", 8, 1, 8, 20, 4, 6, 3, 1),
    ("float", 4, 2, 8, 20, 8, 4, 3, 1),     # 32 x 1280
    ("float", 8, 1, 6, 28, 8, 4, 3, 1),     # 48 x 896
    ("float", 8, 1, 6, 28, 16, 3, 3, 1),
    ("float", 8, 1, 6, 28, 16, 2, 3, 1),
    ("float", 8, 1, 6, 28, 4, 6, 3, 1),
    ("float", 8, 1, 6, 20, 8, 4, 4, 1),     # 48 x 640
    ("float", 8, 1, 4, 28, 8, 4, 4, 1),     # 32 x 896
    ("float", 8, 1, 5, 36, 8, 4, 3, 1),     # 40 x 1152
    ("float", 8, 1, 4, 44, 8, 3, 3, 1),     # 32 x 1408
    ("float", 8, 1, 4, 36, 16, 3, 3, 1),    # 32 x 1152
    # ---- fp32, coarse DM grids: shifts growing by up to 7-8 samples per DM step (q <= 7)
    ("float", 12, 1, 4, 20, 16, 3, 7, 1),   # 48 x 640
    ("float", 12, 1, 4, 20, 8, 4, 7, 1),
    # ---- fp32, small problems (several CTAs per SM)
    ("float", 8, 1, 4, 12, 8, 3, 4, 2),     # 32 x 384, 2 CTAs/SM
    ("float", 4, 1, 4, 12, 8, 3, 4, 4),     # 16 x 384
    # ---- uint8 (16-bit pair counters): TT pairs = 2*TT samples per thread and DM
    ("uint8_t", 12, 1, 4, 28, 8, 3, 4, 1),  # 48 x 1792, 12 warps
    ("uint8_t", 12, 1, 4, 28, 8, 2, 4, 1),
    ("uint8_t", 12, 1, 4, 20, 8, 3, 4, 1),  # 48 x 1280
    ("uint8_t", 12, 1, 4, 20, 16, 3, 4, 1),
    ("uint8_t", 12, 1, 4, 20, 12, 4, 4, 1),
    ("uint8_t", 12, 1, 4, 20, 8, 4, 4, 1),
    ("uint8_t", 12, 1, 4, 28, 16, 2, 4, 1),
    ("uint8_t", 12, 1, 4, 28, 12, 3, 4, 1),
    ("uint8_t", 12, 1, 5, 20, 16, 3, 4, 1),
    ("uint8_t", 16, 1, 5, 12, 16, 3, 4, 1),
    ("uint8_t", 16, 1, 5, 12, 12, 4, 4, 1),
    ("uint8_t", 16, 1, 5, 12, 16, 4, 4, 1),
    ("uint8_t", 16, 1, 5, 12, 24, 2, 4, 1),
    ("uint8_t", 16, 1, 5, 12, 32, 2, 4, 1),
    ("uint8_t", 16, 1, 4, 20, 16, 3, 4, 1),  # 64 x 1280, 16 warps
    ("uint8_t", 16, 1, 4, 20, 12, 4, 4, 1),
    ("uint8_t", 16, 1, 4, 20, 24, 2, 4, 1),
    ("uint8_t", 16, 1, 4, 20, 12, 3, 4, 1),
    ("uint8_t", 16, 1, 4, 12, 16, 3, 4, 1),
    ("uint8_t", 12, 1, 5, 20, 8, 3, 4, 1),  # 60 x 1280
    ("uint8_t", 12, 1, 6, 12, 8, 3, 4, 1),  # 72 x 768
    ("uint8_t", 16, 1, 5, 12, 8, 3, 4, 1),  # 80 x 768, 16 warps
    ("uint8_t", 16, 1, 4, 12, 8, 3, 4, 1),  # 64 x 768
    ("uint8_t", 16, 1, 6, 12, 8, 3, 4, 1),  # 96 x 768
    ("uint8_t", 8, 1, 6, 28, 8, 3, 4, 1),   # 48 x 1792, 8 warps
    ("uint8_t", 8, 1, 8, 20, 8, 3, 4, 1),   # 64 x 1280
    ("uint8_t", 8, 1, 4, 36, 8, 3, 4, 1),   # 32 x 2304
    ("uint8_t", 12, 1, 8, 12, 8, 3, 4, 1),  # 96 x 768
    ("uint8_t", 12, 1, 4, 20, 16, 3, 7, 1), # 48 x 1280, q <= 7 (coarse DM grids)
    ("uint8_t", 4, 1, 4, 12, 8, 3, 4, 4),   # 16 x 768, small problems
    # ---- LAZY = 1 (10th field): upper window quads loaded only on the paths that read them
    ("float", 16, 1, 4, 20, 20, 3, 3, 1, 1),   # 64 x 640
    ("float", 16, 1, 4, 20, 16, 3, 3, 1, 1),
    ("float", 16, 1, 4, 20, 12, 4, 3, 1, 1),
    ("float", 12, 1, 4, 28, 16, 3, 3, 1, 1),   # 48 x 896
    ("float", 12, 1, 4, 28, 12, 4, 3, 1, 1),
    ("float", 12, 1, 5, 20, 16, 3, 3, 1, 1),   # 60 x 640
    ("float", 12, 1, 4, 20, 16, 3, 4, 1, 1),   # 48 x 640, q <= 4
    ("float", 16, 1, 6, 12, 16, 3, 4, 1, 1),   # 96 x 384
    ("float", 16, 1, 4, 12, 16, 3, 4, 1, 1),   # 64 x 384
    ("float", 8, 1, 6, 28, 16, 3, 3, 1, 1),    # 48 x 896, 8 warps
    ("float", 8, 1, 8, 20, 8, 4, 3, 1, 1),     # 64 x 640, 8 warps
    ("float", 12, 1, 4, 20, 16, 3, 7, 1, 1),   # 48 x 640, q <= 7 (coarse DM grids)
    ("float", 8, 1, 4, 12, 8, 3, 4, 2, 1),     # 32 x 384, 2 CTAs/SM (small problems)
    ("uint8_t", 16, 1, 4, 20, 16, 3, 4, 1, 1),  # 64 x 1280
    ("uint8_t", 16, 1, 4, 20, 12, 4, 4, 1, 1),
    ("uint8_t", 16, 1, 4, 20, 12, 3, 4, 1, 1),
    ("uint8_t", 12, 1, 4, 20, 16, 3, 4, 1, 1),  # 48 x 1280
    ("uint8_t", 12, 1, 4, 28, 8, 3, 4, 1, 1),   # 48 x 1792
    ("uint8_t", 12, 1, 5, 20, 16, 3, 4, 1, 1),  # 60 x 1280
    ("uint8_t", 16, 1, 5, 12, 16, 3, 4, 1, 1),  # 80 x 768
    ("uint8_t", 16, 1, 4, 12, 16, 3, 4, 1, 1),  # 64 x 768
    ("uint8_t", 12, 1, 4, 20, 16, 3, 7, 1, 1),  # 48 x 1280, q <= 7
    ("uint8_t", 16, 1, 4, 20, 16, 3, 3, 1, 1),  # 64 x 1280, q <= 3
]


def _combo(t):
    return ("u32" if t[0] == "uint8_t" else "f32", t[3], t[4], t[7], t[9] if len(t) > 9 else 0)


def tree_combos():
    """(element type, DT, TT, QMAX, LAZY) lattices gen_tree.py must emit."""
    return sorted({"%s:%d,%d,%d,%d" % _combo(t) for t in TREE})


def units():
    """[(unit name, C++ expression making the Variant, generated lattice header or None)] in registry
    order: generic, lds, tree."""
    out = []
    for i, t in enumerate(GENERIC):
        out.append(("generic%d" % i, "make_generic<%s>()" % t, None))
    for i, t in enumerate(LDS):
        out.append(("lds%d" % i, "make_tiled<Tile<%s>>()" % ", ".join(str(x) for x in t), None))
    for i, t in enumerate(TREE):
        out.append(("tree%d" % i, "make_tree<TreeTile<%s>>()" % ", ".join(str(x) for x in t),
                    "tree_gen_%s_%d_%d_%d_%d.cuh" % _combo(t)))
    return out
