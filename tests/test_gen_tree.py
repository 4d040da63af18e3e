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


QUAD = r"asm volatile\(\"ld\.shared\.v4\.\w+ \{%0, %1, %2, %3\}, \[%4 \+ (\d+)\];\"[^\n;]*;"


def quads(text):
    """Indices of the 16-byte window quads the ld.shared.v4 statements in `text` load."""
    offs = [int(x) for x in re.findall(QUAD, text)]
    assert all(o % 16 == 0 for o in offs)
    return [o // 16 for o in offs]


def parse_lattice(text, q):
    """Nodes of loop_q<q>: {label: (j, r, tt, quads loaded before the adds, {bit: (next label, quads
    loaded on that edge)} or None for a last-DM node)}, its window length, the quads the channel entry
    loads up front, the m0 entry map, and the slope bit the function loops on."""
    body = text.split("void loop_q%d(" % q)[1].split("OUT:;")[0]
    wlen = int(re.search(r"(?:float|uint32_t) w\[(\d+)\];", body).group(1))
    first = re.search(ENTRY, body)
    upfront = quads(first[1])
    assert upfront == list(range(len(upfront)))                # consecutive quads from the window's start
    entry = {3: first[2], 2: first[3], 1: first[4], 0: first[5]}
    nodes = {}
    pat = (r"N_(\d+)_(\d+):\s*\n((?:\s*asm volatile\(\"ld\.shared[^\n]*\n)*)"
           r"\s*tree_add<(\d+), (\d+)>\(acc\[(\d+)\], w(?:, zero, one)?\);\s*\n"
           r"((?:(?!\s*N_\d+_\d+:).*\n?)*)")
    qbit = None
    for m in re.finditer(pat, body):
        j, r, pre, radd, tt, jacc, tail = int(m[1]), int(m[2]), m[3], int(m[4]), int(m[5]), int(m[6]), m[7]
        assert r == radd and j == jacc
        t = re.match(r"\s*if \(d & (\d+)u\) (?:\{ (.*?) goto (N_\d+_\d+); \}|goto (N_\d+_\d+);) "
                     r"else goto (N_\d+_\d+);", tail)
        if t:
            assert int(t[1]) == 1 << (24 + j)
            nodes["N_%d_%d" % (j, r)] = (j, r, tt, quads(pre),
                                         {1: (t[3] or t[4], quads(t[2] or "")), 0: (t[5], [])})
        else:
            # the loop step: advance, leave on another slope class, reload, re-enter on m0
            st = re.match(r"\s*asm volatile\(\"// step q%d r%d\"\);\s*\n\s*rows \+= lrow_b;\s*\n\s*d = dn;\s*\n"
                          r"\s*if \(!\(d & (\d+)u\)\) goto OUT;\s*\n\s*" % (q, r) + ENTRY, tail)
            assert st, tail[:200]
            assert not pre
            qbit = int(st[1])
            assert {3: st[3], 2: st[4], 1: st[5], 0: st[6]} == entry and st[2] == first[1]
            nodes["N_%d_%d" % (j, r)] = (j, r, tt, [], None)
    return nodes, wlen, upfront, entry, qbit


@pytest.mark.parametrize("dt,tt,qmax,typ,lazy", [
    (4, 28, 3, "f32", 0), (6, 28, 4, "f32", 0), (8, 20, 3, "f32", 0), (4, 12, 4, "f32", 0),
    (4, 28, 4, "u32", 0), (5, 20, 4, "u32", 0),
    (4, 20, 3, "f32", 1), (4, 28, 3, "f32", 1), (5, 20, 7, "f32", 1), (8, 20, 3, "f32", 1),
    (4, 20, 4, "u32", 1), (5, 12, 4, "u32", 1), (6, 28, 4, "u32", 1)])
def test_lattice_walk_visits_the_right_offsets(dt, tt, qmax, typ, lazy):
    """Every path (q, m0, bits) visits the nodes (j, R_j), stays inside the window, and reads only window
    quads that were loaded on THAT path (the lazy lattices load the upper quads on demand), each once."""
    text = gen_tree.emit(dt, tt, qmax, typ, lazy)
    assert "struct TreeStep<%s, %d, %d, %d, %d>" % (gen_tree.CTYPE[typ][0], dt, tt, qmax, lazy) in text
    assert "WNMAX = %d" % gen_tree.wn(dt, tt, qmax) in text
    saved = 0
    for q in range(qmax + 1):
        nodes, wlen, upfront, entry, qbit = parse_lattice(text, q)
        assert wlen == gen_tree.wn(dt, tt, q)
        assert qbit == 0x10000 << q
        if not lazy:
            assert len(upfront) * 4 == wlen
        for m0 in range(4):
            for bits in itertools.product((0, 1), repeat=dt - 1):
                label, r_expect = entry[m0], m0
                loaded = list(upfront)
                for j in range(dt):
                    jn, r, ttn, pre, nxt = nodes[label]
                    assert (jn, r, ttn) == (j, r_expect, tt)
                    assert r + tt <= wlen                      # the add block stays inside the window
                    loaded += pre
                    assert set(range(r // 4, (r + tt - 1) // 4 + 1)) <= set(loaded), (q, m0, bits, j)
                    if j + 1 < dt:
                        label, on_edge = nxt[bits[j]]
                        loaded += on_edge
                        r_expect += q + bits[j]
                    else:
                        assert nxt is None                     # last DM: the loop step follows
                assert len(loaded) == len(set(loaded)), "a quad was loaded twice on one path"
                # nothing loaded that the path does not read, beyond the up-front part
                assert set(loaded) - set(upfront) <= set(range((r_expect + tt - 1) // 4 + 1))
                saved += wlen // 4 - len(loaded)
        # no unreachable or missing nodes: exactly (4 + j) offsets per level
        for j in range(dt):
            assert sorted(r for (jj, r, _, _, _) in nodes.values() if jj == j) == \
                list(range(j * q, j * q + 4 + j))
    assert (saved > 0) == bool(lazy)


def test_chunk_loop_dispatches_one_hot_slope_classes():
    text = gen_tree.emit(4, 28, 3)
    chunk = text.split("void chunk(")[1]
    assert "uint32_t d = tree_desc<0>(ds);" in chunk
    for q in range(4):
        assert "if (d & %du) { loop_q%d<WD>(acc, rows, ds, d, lrow_b); goto NEXT; }" % (0x10000 << q, q) in chunk
    # the uint8 lattices have the same shape (their adds are carry chains: gen_tree.py HEADER)
    text8 = gen_tree.emit(4, 28, 4, "u32")
    assert "loop_q4<WD>(acc, rows, ds, d, lrow_b)" in text8.split("void chunk(")[1]
    assert "tree_add<7, 28>(acc[1], w);" in text8
    assert "add.cc.u32 %0, %0, %2; addc.u32 %1, %1, %3;" in gen_tree.HEADER


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
    assert [u[0] for u in units[:2]] == ["generic0", "generic1"]
    assert len(units) == len(v.GENERIC) + len(v.LDS) + len(v.TREE)
    assert len(set(u[1] for u in units)) == len(units), "duplicate variant"
    build.generate()
    inc = open(os.path.join(build.OBJ, "registry_gen.inc")).read()
    assert [m for m in re.findall(r"^    variant_(\w+),$", inc, flags=re.M)] == [u[0] for u in units]
    for t in v.TREE:
        typ = "u32" if t[0] == "uint8_t" else "f32"
        assert "%s:%d,%d,%d,%d" % (typ, t[3], t[4], t[7], t[9] if len(t) > 9 else 0) in v.tree_combos()
        assert t[4] % 4 == 0 and (t[4] // 4) % 2 == 1, "TT/4 odd keeps LDS.128 conflict-free"
