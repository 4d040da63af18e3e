"""Host-side logic of bench.py that needs no GPU: which on-chip roof a kernel kind is measured against
(DESIGN.md section 6), the DRAM-traffic table under profiles/, and the compulsory-byte count of the
north star's HBM fraction."""
import csv
import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

import bench  # noqa: E402
from paper_1601_01165_b200 import workloads as wl  # noqa: E402


def test_binding_roof_follows_the_kernel_kind():
    mhz = 1965.0
    b, p, _ = bench.binding_roof("tree_f32: 48x896 DMsxsamples/CTA, 4x28 outputs/thread, cc16 s3 q3 b1", wl.APERTIF, mhz)
    assert b == "alu" and p == pytest.approx(148 * 128 * 1.965e9 / 1e12)          # 37.2 T fp32 adds/s
    b, p8, _ = bench.binding_roof("tree_u8: 80x768 DMsxsamples/CTA, 5x24 outputs/thread, cc16 s3 q4 b1", wl.SURVEY8, mhz)
    assert b == "alu" and p8 == pytest.approx(2 * p)                               # two 16-bit counters per add
    b, pl, _ = bench.binding_roof("lds_f32: 16x1024 DMsxsamples/CTA, 4x16 outputs/thread, cc8 s2 b2", wl.LOFAR, mhz)
    assert b == "lds" and pl == pytest.approx(p / 4)                               # 32 words vs 128 lanes per clk
    assert bench.binding_roof("generic_f32: ...", wl.APERTIF, mhz)[0] == "l2"


def test_compulsory_bytes_match_the_survey_table():
    # 273.2 MB, 1673.3 MB, 911.3 MB, 10 929 MB (input once + output once)
    assert bench.compulsory_bytes(wl.APERTIF, 26707) == 1024 * 26707 * 4 + 2048 * 20000 * 4 == 273231872
    assert bench.compulsory_bytes(wl.LOFAR, 272797) == 1673318016
    assert bench.compulsory_bytes(wl.SURVEY8, 68987) == 1536 * 68987 + 4096 * 49152 * 4 == 911270400
    assert bench.compulsory_bytes(wl.BATCH40, 26707) == 40 * 273231872


def test_memory_cap_counts_the_pair_workspace_of_the_uint8_tree_kernels():
    # survey8: 106 MB of input + 805 MB of output per beam, and 1536 x (24576 + 19835 -> 44412) x 4 B = 273 MB of
    # pairs for the tree_u8 kernels only: 152 beams in 180 GB, not the 197 that input + output alone would give
    in_pitch, pair_pitch = 68992, 44412
    io = 1536 * in_pitch + 4096 * 49152 * 4
    tree = bench.resident_bytes_per_beam(wl.SURVEY8, in_pitch, pair_pitch, "tree_u8: 64x1280 ...")
    assert tree == io + 1536 * pair_pitch * 4 and int(180e9 // tree) == 152
    assert bench.resident_bytes_per_beam(wl.SURVEY8, in_pitch, pair_pitch, "lds_u8: 16x1024 ...") == io
    assert int(180e9 // io) == 197
    assert bench.resident_bytes_per_beam(wl.APERTIF, 26708, 0, "tree_f32: 64x640 ...") == 1024 * 26708 * 4 + 2048 * 20000 * 4


def test_traffic_table_names_shipped_winners_and_existing_summaries():
    rows = {r["config"]: r for r in csv.DictReader(open(bench.TRAFFIC_CSV))}
    assert set(rows) == {"apertif", "lofar", "survey8", "batch40"}
    shipped = open(os.path.join(ROOT, "paper_1601_01165_b200", "tuned", "b200.tsv")).read()
    for name, r in rows.items():
        assert r["variant"] in shipped, "the captured variant of %s is not a shipped winner" % name
        assert os.path.exists(os.path.join(ROOT, r["source"].split(" ")[0]))
        # the capture is of the kernel sources as they are now: editing a kernel without a new ncu capture fails here
        assert r["kernel_sources_sha16"] == bench.kernel_sources_sha16(), "re-capture profiles/r03_traffic.csv"
        got, src = bench.ncu_traffic(name, r["variant"])
        assert got == int(r["dram_bytes_per_step"]) and src == r["source"]
        assert bench.ncu_traffic(name, "some other variant")[0] is None
        assert int(r["compulsory_bytes"]) == bench.compulsory_bytes(
            wl.CONFIGS[name], {"apertif": 26707, "lofar": 272797, "survey8": 68987, "batch40": 26707}[name])
    assert bench.ncu_traffic("tiny", "x") == (None, None)


def test_partial_retune_keeps_the_other_entries():
    from paper_1601_01165_b200 import tuning
    old = "k1\tvariant a\t1 ms\nk2\tvariant b\t2 ms\n"
    new = "k2\tvariant c\t1.5 ms\nk3\tvariant d\t3 ms\n"
    assert tuning.merge_entries(old, new) == "k1\tvariant a\t1 ms\nk2\tvariant c\t1.5 ms\nk3\tvariant d\t3 ms\n"
    assert tuning.merge_entries("", new) == new
    shipped = open(tuning.SHIPPED).read()
    assert tuning.merge_entries(shipped, "") == shipped       # unique keys: the five BASELINE configs (apertif
    assert len({l.split("\t")[0] for l in shipped.splitlines()}) == 7   # for 1 and 8 beams) + the paper's two setups
