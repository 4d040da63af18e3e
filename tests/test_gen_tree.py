"""Host logic of the KIND_TREE kernels: the generated add lattice (csrc/gen_tree.py).  The walk
through the generated labels must visit, for every slope class q, window misalignment m0 and increment
bits, exactly the nodes (j, R_j) with R_0 = m0 and R_j = R_{j-1} + q + bit_j, and
every node must stay inside the window the class loads."""
import importlib.util
import itertools
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
spec = importlib.util.spec_from_file_location(
    "gen_tree", os.path.join(ROOT, "paper_1601_01165_b200", "csrc", "gen_tree.py"))
gen_tree = importlib.util.module_from_spec(spec)
spec.loader.exec_module(gen_tree)


ENTRY = (r"dn = tree_desc<WD \* 4>\(ds\);\s*\n\s*ds \+= WD \* 4;\s*\n\s*p = rows \+ \(d & 65520u\);\s*\n"
         r"((?:\s*asm volatile\(\"ld\.shared\.v4[^\n]*\n)+)"
         r"\s*if \(d & 2u\) \{ if \(d & 1u\) goto (\w+); else goto (\w+); \}\s*\n\s*"
         r"else \{ if \(d & 1u\) goto (\w+); else goto (\w+); \}")


def parse_lattice(text, q):
    """Nodes of loop_q<q>: {label: (j, r, tt, {bit value: next label} or the loop step's m0 entry map)},
    its window length, the m0 entry map of the function's entry, and the slope bit it loops on."""
    body = text.split("void loop_q%d(" % q)[1].split("OUT:;")[0]
    wlen = int(re.search(r"(?:float|uint32_t) w\[(\d+)\];", body).group(1))
    first = re.search(ENTRY, body)
    assert len(re.findall(r"ld\.shared\.v4", first[1])) * 4 == wlen
    offs = [int(x) for x in re.findall(r"\[%4 \+ (\d+)\]", first[1])]
    assert offs == list(range(0, 4 * wlen, 16))               # consecutive 16-byte quads
    entry = {3: first[2], 2: first[3], 1: first[4], 0: first[5]}
    nodes = {}
    pat = (r"N_(\d+)_(\d+):\s*\n\s*tree_add<(\d+), (\d+)>\(acc\[(\d+)\], w(?:, zero, one)?\);\s*\n"
           r"((?:(?!\s*N_\d+_\d+:).*\n?)*)")
    qbit = None
    for m in re.finditer(pat, body):
        j, r, radd, tt, jacc, tail = int(m[1]), int(m[2]), int(m[3]), int(m[4]), int(m[5]), m[6]
        assert r == radd and j == jacc
        t = re.match(r"\s*if \(d & (\d+)u\) goto (N_\d+_\d+); else goto (N_\d+_\d+);", tail)
        if t:
            assert int(t[1]) == 1 << (24 + j)
            nodes["N_%d_%d" % (j, r)] = (j, r, tt, {1: t[2], 0: t[3]})
        else:
            # the loop step: advance, leave on another slope class, reload, re-enter on m0
            st = re.match(r"\s*asm volatile\(\"// step q%d r%d\"\);\s*\n\s*rows \+= lrow_b;\s*\n\s*d = dn;\s*\n"
                          r"\s*if \(!\(d & (\d+)u\)\) goto OUT;\s*\n\s*" % (q, r) + ENTRY, tail)
            assert st, tail[:200]
            qbit = int(st[1])
            assert {3: st[3], 2: st[4], 1: st[5], 0: st[6]} == entry and st[2] == first[1]
            nodes["N_%d_%d" % (j, r)] = (j, r, tt, None)
    return nodes, wlen, entry, qbit


@pytest.mark.parametrize("dt,tt,qmax,typ", [(4, 28, 3, "f32"), (6, 28, 4, "f32"), (8, 20, 3, "f32"),
                                            (4, 12, 4, "f32"), (4, 28, 4, "u32"), (5, 20, 4, "u32")])
def test_lattice_walk_visits_the_right_offsets(dt, tt, qmax, typ):
    text = gen_tree.emit(dt, tt, qmax, typ)
    assert "struct TreeStep<%s, %d, %d, %d>" % (gen_tree.CTYPE[typ][0], dt, tt, qmax) in text
    assert "WNMAX = %d" % gen_tree.wn(dt, tt, qmax) in text
    for q in range(qmax + 1):
        nodes, wlen, entry, qbit = parse_lattice(text, q)
        assert wlen == gen_tree.wn(dt, tt, q)
        assert qbit == 0x10000 << q
        for m0 in range(4):
            for bits in itertools.product((0, 1), repeat=dt - 1):
                label, r_expect = entry[m0], m0
                for j in range(dt):
                    jn, r, ttn, nxt = nodes[label]
                    assert (jn, r, ttn) == (j, r_expect, tt)
                    assert r + tt <= wlen                      # the add block stays inside the window
                    if j + 1 < dt:
                        label = nxt[bits[j]]
                        r_expect += q + bits[j]
                    else:
                        assert nxt is None                     # last DM: the loop step follows
        # no unreachable or missing nodes: exactly (4 + j) offsets per level
        for j in range(dt):
            assert sorted(r for (jj, r, _, _) in nodes.values() if jj == j) == \
                list(range(j * q, j * q + 4 + j))


def test_chunk_loop_dispatches_one_hot_slope_classes():
    text = gen_tree.emit(4, 28, 3)
    chunk = text.split("void chunk(")[1]
    assert "uint32_t d = tree_desc<0>(ds);" in chunk
    for q in range(4):
        assert "if (d & %du) { loop_q%d<WD>(acc, rows, ds, d, lrow_b); goto NEXT; }" % (0x10000 << q, q) in chunk
    # the uint8 lattices carry the two run-time constants that pin the pipe of each add
    text8 = gen_tree.emit(4, 28, 4, "u32")
    assert "loop_q4<WD>(acc, rows, ds, d, lrow_b, zero, one)" in text8.split("void chunk(")[1]
    assert "tree_add<7, 28>(acc[1], w, zero, one);" in text8


def test_descriptor_layout_constants():
    """gen_tree.py and desc_kernel (shift_table.cu) agree on the descriptor word."""
    assert (gen_tree.Q_SHIFT, gen_tree.BIT_SHIFT, gen_tree.OFF_MASK) == (16, 24, 0xfff0)
    src = open(os.path.join(ROOT, "paper_1601_01165_b200", "csrc", "shift_table.cu")).read()
    assert "bits << 24 | (0x10000u << q) | (w >> 2) << 4 | (w & 3u)" in src


def test_variant_list_is_the_single_source_of_the_registry():
    """csrc/variants.py is the one place a variant is added: the generated registry
    has one maker per entry, in list order, generic first."""
    from paper_1601_01165_b200 import build
    v = build._variants()
    units = v.units()
    assert [n for n, _ in units[:2]] == ["generic0", "generic1"]
    assert len(units) == len(v.GENERIC) + len(v.LDS) + len(v.TREE)
    assert len(set(e for _, e in units)) == len(units), "duplicate variant"
    build.generate()
    inc = open(os.path.join(build.OBJ, "registry_gen.inc")).read()
    assert [m for m in re.findall(r"^    variant_(\w+),$", inc, flags=re.M)] == [n for n, _ in units]
    for t in v.TREE:
        typ = "u32" if t[0] == "uint8_t" else "f32"
        assert "%s:%d,%d,%d" % (typ, t[3], t[4], t[7]) in v.tree_combos()
        assert t[4] % 4 == 0 and (t[4] // 4) % 2 == 1, "TT/4 odd keeps LDS.128 conflict-free"
