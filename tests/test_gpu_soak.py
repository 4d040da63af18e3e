"""Soak tests in place of a race detector (compute-sanitizer's racecheck cannot run on this pool, DESIGN.md
section 11): every staged kernel (tree_f32, tree_u8, lds_*) runs 30 times back to back on two alternating
streams on a shape that gives every persistent CTA several tiles over two beams, a ragged last chunk for
every stage depth and ragged DM and time tiles.  All 30 outputs must be bit-identical to the first, and the
first must meet the oracle.  A missing proxy fence or barrier phase slip in the mbarrier / bulk-copy rings
(the bug of commit 2840de6) shows up as a run that differs.  Also: one uint8 plan on two streams without any
ordering by the caller (include/dedisp.h: the library hands the pair workspace from stream to stream), and
full-size repeats of the two fp32 headline configs."""
import numpy as np
import pytest

import oracle
from paper_1601_01165_b200 import workloads as wl
from test_gpu_parity import TOL, check_full, dd, make_case, out_buffer, to_host  # noqa: F401

pytestmark = pytest.mark.gpu

RUNS = 30

# 70 channels = 3 x 20 + 10 = 4 x 16 + 6 = 5 x 12 + 10 = 8 x 8 + 6: a ragged last chunk for every stage depth;
# 900 DMs and 12001 samples are multiples of no tile; 64x640 tiles: 15 x 19 x 2 beams = 570 tiles = 3.9 per SM
SOAK_F32 = wl.scaled(wl.APERTIF, name="soak_f32", nr_channels=70, channel_bw_MHz=300.0 / 70, nr_dms=900,
                     nr_samples=12001, nr_beams=2)
SOAK_U8 = wl.scaled(wl.SURVEY8, name="soak_u8", nr_channels=70, channel_bw_MHz=300.0 / 70, nr_dms=900,
                    nr_samples=24002, nr_beams=2)
# LOFAR-like band: long shifts, the shapes the lds kernels win
SOAK_LDS = wl.scaled(wl.LOFAR, name="soak_lds", nr_channels=22, channel_bw_MHz=6.0 / 22, nr_dms=300,
                     nr_samples=30001, nr_beams=2)


def soak(dd, setup, prefixes):
    import torch
    plan, table, x, d_in = make_case(dd, setup)
    exact = setup.in_dtype == wl.U8
    ref, sabs = oracle.dedisperse(x, table, setup.nr_samples, want_sabs=True)
    streams = [torch.cuda.Stream(), torch.cuda.Stream()]
    fill = -1 if exact else float("nan")
    outs = [out_buffer(setup, fill=fill) for _ in range(RUNS)]
    ran = 0
    for v in plan.supported_variants():
        name = dd.variant_name(v)
        if not name.startswith(prefixes):
            continue
        for o in outs:
            o.fill_(fill)
        plan.execute_variant(v, d_in, outs[0])      # first use prepares the variant (may allocate)
        torch.cuda.synchronize()
        for i in range(1, RUNS):                    # no synchronisation between the runs
            plan.execute_variant(v, d_in, outs[i], nr_beams=setup.nr_beams, stream=streams[i % 2])
        torch.cuda.synchronize()
        outs[0].fill_(fill)
        plan.execute_variant(v, d_in, outs[0], nr_beams=setup.nr_beams)
        torch.cuda.synchronize()
        for i in range(1, RUNS):
            # bit patterns compared as integers: NaN-poisoned remnants would not equal themselves as floats
            assert torch.equal(outs[i].view(torch.int32), outs[0].view(torch.int32)), "%s: run %d differs" % (name, i)
        try:
            check_full(setup, to_host(setup, outs[0]), ref, sabs, exact)
        except AssertionError as e:
            raise AssertionError("%s on %s: %s" % (name, setup.name, e))
        ran += 1
    plan.destroy()
    return ran


def test_soak_every_fp32_tree_variant(dd):
    assert soak(dd, SOAK_F32, ("tree_f32",)) >= 30


def test_soak_every_uint8_tree_variant(dd):
    assert soak(dd, SOAK_U8, ("tree_u8",)) >= 10


def test_soak_every_lds_variant(dd):
    assert soak(dd, SOAK_LDS, ("lds_f32",)) >= 5
    assert soak(dd, wl.scaled(SOAK_LDS, name="soak_lds_u8", in_dtype=wl.U8, values="u8"), ("lds_u8",)) >= 2


def test_one_uint8_plan_on_two_streams_without_ordering_by_the_caller(dd):
    """include/dedisp.h: tree_u8 calls on one plan share its pair workspace and the library orders them itself.
    20 interleaved calls on two streams, four different inputs, no events, no synchronisation: every output
    equals the oracle's."""
    import torch
    s = wl.scaled(wl.SURVEY8, name="two_streams", nr_channels=512, channel_bw_MHz=300.0 / 512, nr_dms=512,
                  nr_samples=20000)
    plan, table, x0, d0 = make_case(dd, s)
    tree = [v for v in plan.supported_variants() if dd.variant_name(v).startswith("tree_u8")]
    plan.set_variant(tree[0])
    xs, dins, refs = [x0], [d0], [oracle.dedisperse(x0, table, s.nr_samples)]
    for k in range(1, 4):
        x = wl.make_input(wl.scaled(s, seed=s.seed + 100 * k), plan.in_samples, plan.in_pitch)
        xs.append(x)
        dins.append(torch.from_numpy(x).cuda())
        refs.append(oracle.dedisperse(x, table, s.nr_samples))
    streams = [torch.cuda.Stream(), torch.cuda.Stream()]
    outs = [out_buffer(s, fill=-1) for _ in range(20)]
    torch.cuda.synchronize()
    for i in range(20):
        plan.execute(dins[(i * 3) % 4], outs[i], stream=streams[i % 2])
    torch.cuda.synchronize()
    for i in range(20):
        assert np.array_equal(to_host(s, outs[i]).astype(np.uint64), refs[(i * 3) % 4]), "call %d" % i
    plan.destroy()


@pytest.mark.parametrize("name,beams", [("apertif", 1), ("batch40", 40)])
def test_full_size_repeats_are_bit_identical(dd, name, beams):
    """The shipped winner at full size, 10 runs back to back on two streams: identical bits (parity of one run
    against the oracle at this size is test_gpu_parity's job)."""
    import torch
    from paper_1601_01165_b200 import tuning
    s = wl.CONFIGS[name]
    with dd.Plan(*s.plan_args()) as plan:
        tuning.apply_shipped(plan, nr_beams=beams)
        gen = torch.Generator(device="cuda").manual_seed(s.seed)
        d_in = torch.randn((beams, s.nr_channels, plan.in_pitch), dtype=torch.float32, device="cuda", generator=gen)
        first = torch.empty((beams, s.nr_dms, s.nr_samples), dtype=torch.float32, device="cuda")
        nxt = [torch.empty_like(first), torch.empty_like(first)]
        streams = [torch.cuda.Stream(), torch.cuda.Stream()]
        plan.execute(d_in, first, nr_beams=beams)
        torch.cuda.synchronize()
        for i in range(1, 10, 2):
            for k in range(2):
                nxt[k].fill_(float("nan"))
            torch.cuda.synchronize()
            for k in range(2):
                plan.execute(d_in, nxt[k], nr_beams=beams, stream=streams[k])
            torch.cuda.synchronize()
            for k in range(2):
                assert torch.equal(nxt[k].view(torch.int32), first.view(torch.int32)), "run %d" % (i + k)
