"""gen_tree.py -- build-time generator of the KIND_TREE inner loop (step a5).

The paper generates its kernel source per parameter set at run time; here the one
piece that cannot be expressed with templates is generated at build time: a branch LATTICE that
adds a thread's register window into its DT x TT accumulators with every register index static.

For one channel a thread owns DT adjacent DMs x TT consecutive samples.  The shifts of its DMs are
e_0 <= e_1 <= ... and, because shift(c, dm) is a rounded linear function of the DM index, every
increment e_j - e_{j-1} is q or q+1 for one q per (channel, DM group) (checked at plan creation;
plans that violate it do not get this kernel).  The thread loads the window
w[0 .. WN_q) = row[a0 .. a0 + WN_q) once (LDS.128, a0 16-byte aligned) and DM j adds
w[R_j + k], k < TT, with R_0 = m0 = (e_0 - row origin) & 3 and R_j = R_{j-1} + q + b_j.  m0, q and
the bits b_j are warp-uniform, so the selection is a walk through nodes N[q][j][R] joined by uniform
two-way branches: one test per DM, no indirect jump, no dynamic register index.  Per (DT, TT, QMAX)
the generator emits one lattice function per q and the channel loop of a staged chunk around them.

Two element types: "f32" (fp32 input: float accumulators, FADD / packed FADD2) and "u32" (uint8 input
staged as pairs of 16-bit counters in one 32-bit word, kernel_tree.cuh: one integer add does two adds
whatever the offset).

Usage: python gen_tree.py OUTDIR TYPE:DT,TT,QMAX,LAZY [TYPE:DT,TT,QMAX,LAZY ...]
"""
from __future__ import annotations

import os
import sys


def wn(dt: int, tt: int, q: int) -> int:
    """Window registers for slope class q: offsets reach 3 + (dt-1)*(q+1), rounded to 16 bytes."""
    return (3 + (dt - 1) * (q + 1) + tt + 3) // 4 * 4


CTYPE = {"f32": ("float", "f32", "f"), "u32": ("uint32_t", "u32", "r")}

# Descriptor word of one (channel, DM group), built by desc_kernel (shift_table.cu):
#   [15:4] index of the 16-byte quad of the staged row the group's window starts in, so that
#          d & 0xfff0 is the window's byte offset;  [1:0] m0, the first DM's offset inside that quad;
#   [23:16] one-hot slope class, 0x10000 << q_c;  [31:24] bits, the group's increments being q_c + bit_j.
# A descriptor with no slope bit (0) ends the chunk: the row after a chunk's last channel holds zeros.
Q_SHIFT, BIT_SHIFT, OFF_MASK = 16, 24, 0xfff0


def need(r: int, tt: int) -> int:
    """Highest 16-byte quad of the window a DM at offset r reads (w[r .. r+tt))."""
    return (r + tt - 1) // 4


def first_lazy(tt: int, q: int) -> int:
    """LAZY lattices: quads below this index are loaded when a channel starts, the others only on the
    paths that read them.  No first or second DM of a group ever reads a lazy quad (their offsets are at
    most 3 and 4 + q), so a lazy quad is always requested at least one add block ahead of its use."""
    return need(4 + q, tt) + 1


def emit(dt: int, tt: int, qmax: int, typ: str = "f32", lazy: int = 0) -> str:
    o = []
    wnmax = wn(dt, tt, qmax)
    ct, pt, rc = CTYPE[typ]
    o.append("template <> struct TreeStep<%s, %d, %d, %d, %d> {" % (ct, dt, tt, qmax, lazy))
    o.append("    static constexpr int WNMAX = %d;" % wnmax)
    # One function per slope class q: the channel loop over a run of channels of that class.  The loop
    # has no head block.  Every node of the last DM ends with the loop's step: advance to the next
    # channel, leave if its slope class differs (or it is the chunk's terminator), fetch the descriptor
    # after it, issue the next channel's window loads, and branch on m0 straight to that channel's first
    # node.  So the window loads are in flight while the branches resolve, and a channel costs about
    # three taken branches instead of five.
    #
    # LAZY = 1: shared memory is what binds these kernels, and a quarter of the window words loaded up
    # front are never read: the window is sized for the largest offset the last DM can reach
    # (3 + (DT-1)(q+1)), the typical path stops short of it.  So only the quads below first_lazy() are
    # loaded when the channel starts; node (j, R) requests the quads its successors read and the path so
    # far has not: those both successors need at the node's start, the one only the bit = 1 successor
    # needs on that edge.  Invariant: entering node (j, R), the quads loaded are exactly the up-front ones
    # plus the lazy ones up to need(R); it depends on R alone, not on the path.
    for q in range(qmax + 1):
        n = wn(dt, tt, q)
        qbit = 1 << (Q_SHIFT + q)
        nq = n // 4
        upfront = min(nq, first_lazy(tt, q)) if lazy else nq
        loads = []
        for m in range(nq):
            loads.append('asm volatile("ld.shared.v4.%s {%%0, %%1, %%2, %%3}, [%%4 + %d];" : "=%s"(w[%d]), '
                         '"=%s"(w[%d]), "=%s"(w[%d]), "=%s"(w[%d]) : "r"(p));'
                         % (pt, 16 * m, rc, 4 * m, rc, 4 * m + 1, rc, 4 * m + 2, rc, 4 * m + 3))
        enter = ["dn = tree_desc<WD * 4>(ds);", "ds += WD * 4;", "p = rows + (d & %du);" % OFF_MASK] + \
            loads[:upfront] + [
            "if (d & 2u) { if (d & 1u) goto N_0_3; else goto N_0_2; }",
            "else { if (d & 1u) goto N_0_1; else goto N_0_0; }"]
        o.append("    // slope class q = %d: window of %d registers%s.  rows, ds: shared-memory byte addresses of the"
                 % (q, n, ", quads %d.. on demand" % upfront if upfront < nq else ""))
        o.append("    // thread's place in the current channel's staged row and of the warp's descriptor of that")
        o.append("    // channel; d: that descriptor (warp-uniform).  Returns at the first channel of another class.")
        o.append("    template <int WD>")
        o.append("    static __device__ __forceinline__ void loop_q%d(%s (&acc)[%d][%d], uint32_t &rows, "
                 "uint32_t &ds, uint32_t &d, uint32_t lrow_b) {" % (q, ct, dt, tt))
        o.append("        %s w[%d];" % (ct, n))
        o.append("        uint32_t dn, p;")
        for line in enter:
            o.append("        " + line)
        for j in range(dt):
            for r in range(j * q, j * q + 3 + j + 1):
                o.append("    N_%d_%d:" % (j, r))
                if j + 1 < dt:
                    have = max(upfront - 1, need(r, tt))          # highest quad loaded on entry
                    both = range(have + 1, need(r + q, tt) + 1)    # read by both successors
                    edge = range(max(have, need(r + q, tt)) + 1, need(r + q + 1, tt) + 1)  # by bit = 1 only
                    for m in both:
                        o.append("        " + loads[m])
                    o.append("        tree_add<%d, %d>(acc[%d], w);" % (r, tt, j))
                    if len(edge):
                        o.append("        if (d & %du) { %s goto N_%d_%d; } else goto N_%d_%d;"
                                 % (1 << (BIT_SHIFT + j), " ".join(loads[m] for m in edge), j + 1, r + q + 1,
                                    j + 1, r + q))
                    else:
                        o.append("        if (d & %du) goto N_%d_%d; else goto N_%d_%d;"
                                 % (1 << (BIT_SHIFT + j), j + 1, r + q + 1, j + 1, r + q))
                else:
                    o.append("        tree_add<%d, %d>(acc[%d], w);" % (r, tt, j))
                    # the loop step, one copy per last node (the comment keeps the copies from being
                    # merged back into one shared block behind a jump)
                    o.append('        asm volatile("// step q%d r%d");' % (q, r))
                    o.append("        rows += lrow_b;")
                    o.append("        d = dn;")
                    o.append("        if (!(d & %du)) goto OUT;" % qbit)
                    for line in enter:
                        o.append("        " + line)
        o.append("    OUT:;")
        o.append("    }")
    # the channel loop of one staged chunk.  Testing single bits of a one-hot mask keeps the dispatch
    # compare-and-branch (a chain of q == k tests with five or more cases is turned into an indirect jump
    # through a constant-memory table, LDC + BRX).  No channel counter: the zero descriptor after the
    # chunk's last channel fails every slope test.
    o.append("    // rows: shared-memory byte address of the thread's position in channel 0's staged row;")
    o.append("    // ds: shared-memory byte address of the warp's descriptor of channel 0 (WD words per channel,")
    o.append("    // a zero row after the last channel); lrow_b: bytes per staged row.")
    o.append("    template <int WD>")
    o.append("    static __device__ __forceinline__ void chunk(%s (&acc)[%d][%d], uint32_t rows, "
             "uint32_t ds, uint32_t lrow_b) {" % (ct, dt, tt))
    o.append("        uint32_t d = tree_desc<0>(ds);")
    o.append("    NEXT:")
    for q in range(qmax + 1):
        o.append("        if (d & %du) { loop_q%d<WD>(acc, rows, ds, d, lrow_b); goto NEXT; }"
                 % (1 << (Q_SHIFT + q), q))
    o.append("    }")
    o.append("};")
    return "\n".join(o)


HEADER = """// GENERATED by gen_tree.py -- do not edit.  KIND_TREE add lattices (see gen_tree.py).
#pragma once
#include <stdint.h>
namespace dedisp {
template <typename E, int DT, int TT, int QMAX, int LAZY> struct TreeStep;
// descriptor of one (channel, DM group): a shared-memory load whose address (a 32-bit shared-window
// byte address plus a constant) is the same for the whole warp.
template <int OFF>
__device__ __forceinline__ uint32_t tree_desc(uint32_t p) {
    uint32_t v;
    asm volatile("ld.shared.u32 %0, [%1 + %2];" : "=r"(v) : "r"(p), "n"(OFF));
    return v;
}
// acc[k] += w[R + k], all indices static.  Inline asm keeps the optimiser from merging the add
// blocks of sibling lattice nodes into one block fed by register moves (a MOV costs the issue slot
// the FADD was meant to use).
template <int R, int TT, int WN>
__device__ __forceinline__ void tree_add(float (&acc)[TT], const float (&w)[WN]) {
    static_assert(R + TT <= WN, "window too short");
    if constexpr (R % 2 == 0 && TT % 2 == 0) {
        // even offset: window pairs and accumulator pairs are both 64-bit aligned register pairs,
        // so one packed add (SASS FADD2) does two adds in one issue slot
#pragma unroll
        for (int k = 0; k < TT; k += 2)
            asm volatile(
                "{.reg .b64 a, b; mov.b64 a, {%0, %1}; mov.b64 b, {%2, %3}; add.f32x2 a, a, b; "
                "mov.b64 {%0, %1}, a;}"
                : "+f"(acc[k]), "+f"(acc[k + 1])
                : "f"(w[R + k]), "f"(w[R + k + 1]));
    } else {
#pragma unroll
        for (int k = 0; k < TT; ++k)
            asm volatile("add.f32 %0, %0, %1;" : "+f"(acc[k]) : "f"(w[R + k]));
    }
}
// uint8 input: acc and w hold two 16-bit counters / samples per word, so one 32-bit add does two adds
// whatever the offset.  Integer adds issue at half rate on either of two pipes: IADD3 on the integer
// pipe, IMAD on the FMA pipe.  Left to itself ptxas turns three of four plain adds into IMAD.IADD (84
// lanes/clk/SM measured).  Writing two neighbouring adds as ONE carry chain (add.cc / addc) pins one to
// each pipe, IADD3 + IMAD.X, at 116 lanes/clk/SM (profiles/r02_microbench.md, run 5), without the two
// run-time constants an earlier version needed to keep ptxas from rewriting the adds.  The carry is
// always zero: a word's upper counter stays below 2^16 between flushes, so the low add cannot overflow
// (only lanes past the staged data can, and what they and their right neighbours compute is never stored).
template <int R, int TT, int WN>
__device__ __forceinline__ void tree_add(uint32_t (&acc)[TT], const uint32_t (&w)[WN]) {
    static_assert(R + TT <= WN && TT % 2 == 0, "window too short");
#pragma unroll
    for (int k = 0; k < TT; k += 2)
        asm volatile("add.cc.u32 %0, %0, %2; addc.u32 %1, %1, %3;"
                     : "+r"(acc[k]), "+r"(acc[k + 1]) : "r"(w[R + k]), "r"(w[R + k + 1]));
}
"""


def combo_file(typ, dt, tt, qmax, lazy):
    return "tree_gen_%s_%d_%d_%d_%d.cuh" % (typ, dt, tt, qmax, lazy)


def _write_if_changed(path, text):
    try:
        if open(path).read() == text:
            return
    except OSError:
        pass
    with open(path, "w") as f:
        f.write(text)


def main(argv):
    """Writes OUTDIR/tree_gen_common.cuh and one OUTDIR/tree_gen_<combo>.cuh per lattice (a unit includes
    only its own, so changing one lattice recompiles one unit).  Files whose text is unchanged keep their
    timestamps."""
    outdir = argv[1]
    combos = sorted({(a.split(":")[0],) + tuple(int(x) for x in a.split(":")[1].split(","))
                     for a in argv[2:]})
    _write_if_changed(os.path.join(outdir, "tree_gen_common.cuh"), HEADER + "}  // namespace dedisp\n")
    for typ, dt, tt, qmax, lazy in combos:
        _write_if_changed(os.path.join(outdir, combo_file(typ, dt, tt, qmax, lazy)),
                          "// GENERATED by gen_tree.py -- do not edit.\n#pragma once\n"
                          '#include "tree_gen_common.cuh"\nnamespace dedisp {\n'
                          + emit(dt, tt, qmax, typ, lazy) + "\n}  // namespace dedisp\n")


if __name__ == "__main__":
    main(sys.argv)
