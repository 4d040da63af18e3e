"""GPU edge cases through the C-ABI: ragged / degenerate shapes, alignment, errors, tuner."""
import os

import numpy as np
import pytest

import oracle
from paper_1601_01165_b200 import workloads as wl
from test_gpu_parity import TOL, check_full, dd, make_case, out_buffer, to_host  # noqa: F401

pytestmark = pytest.mark.gpu


def run_all(dd, setup, exact=None):
    plan, table, x, d_in = make_case(dd, setup)
    ref, sabs = oracle.dedisperse(x, table, setup.nr_samples, want_sabs=True)
    exact = (setup.in_dtype == wl.U8 or setup.values == "int16") if exact is None else exact
    for v in plan.supported_variants():
        d_out = out_buffer(setup, fill=-1 if setup.in_dtype == wl.U8 else float("nan"))
        plan.execute_variant(v, d_in, d_out, nr_beams=setup.nr_beams)
        try:
            check_full(setup, to_host(setup, d_out), ref, sabs, exact)
        except AssertionError as e:
            raise AssertionError("%s on %s: %s" % (dd.variant_name(v), setup.name, e))
    plan.destroy()


EDGES = [
    wl.Setup("one_of_each", 1, 1400.0, 1.0, 1000.0, 1, 0.0, 1.0, 1, values="int16", seed=1),
    wl.Setup("one_channel", 1, 300.0, 5.0, 5000.0, 700, 0.0, 2.0, 9, values="int16", seed=2),
    wl.Setup("one_dm", 40, 1400.0, 2.0, 10000.0, 1300, 3.0, 0.0, 1, seed=3),
    wl.Setup("s_not_mult_of_4", 24, 1400.0, 4.0, 20000.0, 1021, 0.0, 0.5, 37, seed=4),
    wl.Setup("s_odd_u8", 24, 1400.0, 4.0, 20000.0, 1021, 0.0, 0.5, 37, in_dtype=wl.U8, values="u8", seed=5),
    wl.Setup("zero_dm_step", 64, 1400.0, 1.0, 20000.0, 2000, 5.0, 0.0, 33, seed=6),   # perfect reuse
    wl.Setup("all_zero_dm", 64, 1400.0, 1.0, 20000.0, 2000, 0.0, 0.0, 16, values="int16", seed=7),
    wl.Setup("few_samples", 48, 1400.0, 1.0, 20000.0, 5, 0.0, 0.25, 130, seed=8),
    wl.Setup("max_u8", 1536, 1220.0, 300.0 / 1536, 24414.0, 64, 0.0, 0.2, 8, in_dtype=wl.U8, values="u8", seed=9),
    wl.Setup("beams3", 20, 1400.0, 3.0, 20000.0, 900, 0.0, 0.25, 50, nr_beams=3, seed=10),
    wl.Setup("beams3_u8", 20, 1400.0, 3.0, 20000.0, 900, 0.0, 0.25, 50, nr_beams=3, in_dtype=wl.U8, values="u8", seed=11),
    wl.Setup("big_steps", 16, 140.0, 0.2, 100000.0, 3000, 0.0, 0.05, 40, seed=12),    # LOFAR-like long shifts
    wl.Setup("dm_first_nonzero", 32, 1420.0, 1.0, 20000.0, 1500, 100.0, 0.25, 45, seed=13),
    # uint8 pair layout: S/2 not a multiple of 4, fewer samples than one pair quad, one DM, and more than
    # 512 channels (three counter flushes) on ragged tiles
    wl.Setup("u8_one_sample", 9, 1400.0, 3.0, 20000.0, 1, 0.0, 0.25, 3, in_dtype=wl.U8, values="u8", seed=14),
    wl.Setup("u8_s6", 20, 1400.0, 3.0, 20000.0, 6, 0.0, 0.25, 21, in_dtype=wl.U8, values="u8", seed=15),
    wl.Setup("u8_one_dm", 40, 1400.0, 2.0, 10000.0, 1303, 3.0, 0.0, 1, in_dtype=wl.U8, values="u8", seed=16),
    wl.Setup("u8_flush3", 700, 1220.0, 300.0 / 700, 24414.0, 1502, 0.0, 0.2, 37, in_dtype=wl.U8, values="u8", seed=17),
]


@pytest.mark.parametrize("setup", EDGES, ids=[s.name for s in EDGES])
def test_edge_shapes_every_variant(dd, setup):
    run_all(dd, setup)


def test_max_u8_value_saturation_is_exact(dd):
    """All-255 input over 1536 channels: every output is 1536*255 = 391680 (fits uint32)."""
    import torch
    s = wl.Setup("all255", 1536, 1220.0, 300.0 / 1536, 24414.0, 300, 0.0, 0.2, 20, in_dtype=wl.U8)
    with dd.Plan(*s.plan_args()) as plan:
        d_in = torch.full((1, s.nr_channels, plan.in_pitch), 255, dtype=torch.uint8, device="cuda")
        for v in plan.supported_variants():
            d_out = out_buffer(s, fill=-1)
            plan.execute_variant(v, d_in, d_out)
            assert (d_out == 1536 * 255).all(), dd.variant_name(v)


def test_execute_is_repeatable_and_stream_ordered(dd):
    import torch
    s = wl.scaled(wl.APERTIF, name="rep", nr_channels=64, channel_bw_MHz=300.0 / 64, nr_dms=64,
                  nr_samples=2000)
    plan, table, x, d_in = make_case(dd, s)
    a, b = out_buffer(s, fill=float("nan")), out_buffer(s, fill=float("nan"))
    st = torch.cuda.Stream()
    plan.execute(d_in, a)
    with torch.cuda.stream(st):
        plan.execute(d_in, b, stream=st)
    torch.cuda.synchronize()
    assert torch.equal(a, b)
    plan.destroy()


@pytest.mark.parametrize("kind", ["tree_f32", "lds_f32"])
def test_two_live_plans_of_different_size_on_one_variant(dd, kind):
    """The large-shared-memory attribute belongs to the kernel, not to a plan: selecting the variant for a
    second plan with shorter staged rows must not lower it under the first plan (whose launch then failed
    with 'invalid argument')."""
    big = wl.scaled(wl.APERTIF, name="two_big", nr_channels=96, channel_bw_MHz=300.0 / 96, nr_dms=700,
                    nr_samples=3000, values="int16")
    small = wl.scaled(big, name="two_small", nr_dms=64, dm_step=0.02)
    pa, ta, xa, da = make_case(dd, big)
    va = [v for v in pa.supported_variants() if dd.variant_name(v).startswith(kind)]
    pb, tb, xb, db = make_case(dd, small)
    common = [v for v in va if pb.variant_supported(v)]
    assert common
    pa.set_variant(common[-1])
    pb.set_variant(common[-1])     # smaller shift span: fewer bytes of dynamic shared memory
    for s, plan, x, table, d_in in ((big, pa, xa, ta, da), (small, pb, xb, tb, db), (big, pa, xa, ta, da)):
        d_out = out_buffer(s, fill=float("nan"))
        plan.execute(d_in, d_out)
        assert np.array_equal(to_host(s, d_out).astype(np.float64), oracle.dedisperse(x, table, s.nr_samples))
    pa.destroy()
    pb.destroy()


@pytest.mark.parametrize("u8", [False, True])
def test_first_execute_of_a_fresh_plan_can_be_captured_into_a_cuda_graph(dd, u8):
    """dedisp_execute promises no allocation, no host sync and no function-attribute call (all done
    when the variant is selected): the FIRST call on a fresh plan is captured into a CUDA graph and
    the replays are bit-exact against the oracle (include/dedisp.h)."""
    import torch
    s = wl.scaled(wl.SURVEY8 if u8 else wl.APERTIF, name="graph", nr_channels=300,
                  channel_bw_MHz=300.0 / 300, nr_dms=150, nr_samples=4100, nr_beams=2,
                  values="u8" if u8 else "int16", in_dtype=wl.U8 if u8 else wl.F32)
    plan, table, x, d_in = make_case(dd, s)
    # a kernel that needs everything a selection prepares: > 48 KB of dynamic shared memory, a
    # descriptor table and (uint8) the pair workspace
    tree = [v for v in plan.supported_variants() if dd.variant_name(v).startswith("tree_")]
    plan.set_variant(tree[0])
    if u8:
        plan.reserve(s.nr_beams)
    ref = oracle.dedisperse(x, table, s.nr_samples)
    d_out = out_buffer(s, fill=-1)
    st = torch.cuda.Stream()
    graph = torch.cuda.CUDAGraph()
    torch.cuda.synchronize()
    with torch.cuda.graph(graph, stream=st):
        plan.execute(d_in, d_out, nr_beams=s.nr_beams, stream=torch.cuda.current_stream())
    for _ in range(2):
        d_out.fill_(-1)
        graph.replay()
        torch.cuda.synchronize()
        got = to_host(s, d_out)
        assert np.array_equal(got.astype(np.uint64 if u8 else np.float64), ref)
    plan.destroy()


def test_u8_batches_larger_than_the_reserved_workspace(dd):
    """A uint8 plan reserves its pair workspace for one beam; a larger batch goes through it one group
    at a time, and after dedisp_plan_reserve in one launch: same bits either way."""
    import torch
    s = wl.Setup("resv", 40, 1400.0, 3.0, 20000.0, 2100, 0.0, 0.25, 70, nr_beams=5, in_dtype=wl.U8,
                 values="u8", seed=21)
    plan, table, x, d_in = make_case(dd, s)
    ref = oracle.dedisperse(x, table, s.nr_samples)
    tv = [v for v in plan.supported_variants() if dd.variant_name(v).startswith("tree_u8")]
    lds = [v for v in plan.supported_variants() if dd.variant_name(v).startswith("lds_u8")]
    assert tv and lds
    # only the variants that run pay for the workspace: a fresh plan on a tree_u8 kernel holds one beam of
    # it, a plan on another kernel none until a tree_u8 variant is selected
    is_tree = dd.variant_name(plan.variant).startswith("tree_u8")
    assert plan.reserved_beams == (1 if is_tree else 0)
    with dd.Plan(*s.plan_args()) as other:
        other.set_variant(lds[0])
        held = other.reserved_beams
        other.set_variant(tv[0])
        assert held in (0, 1) and other.reserved_beams == 1 and other.pair_pitch > s.nr_samples // 2
    plan.set_variant(tv[0])
    assert plan.reserved_beams == 1
    for resv in (1, 2, 5):
        plan.reserve(resv)
        assert plan.reserved_beams == max(resv, 1)
        d_out = out_buffer(s, fill=-1)
        plan.execute_variant(tv[0], d_in, d_out, nr_beams=s.nr_beams)
        assert np.array_equal(to_host(s, d_out).astype(np.uint64), ref), "reserved %d" % resv
    with dd.Plan(*wl.TINY.plan_args()) as f32:
        f32.reserve(4)
        assert f32.reserved_beams == 0      # fp32 plans have no workspace
    plan.destroy()


def test_execute_on_another_device_is_refused(dd):
    """The plan belongs to the device it was created on: with one GPU this can only check
    that the current device is accepted and that the plan reports a mismatch cleanly if there are two."""
    import torch
    s = wl.TINY
    plan, table, x, d_in = make_case(dd, s)
    d_out = out_buffer(s)
    plan.execute(d_in, d_out)
    if torch.cuda.device_count() > 1:
        with torch.cuda.device(1):
            with pytest.raises(dd.DedispError) as e:
                plan.execute(d_in, d_out)
            assert e.value.status == 1
    plan.destroy()


def test_execute_host_matches_device_path(dd):
    import torch
    s = wl.scaled(wl.APERTIF, name="host", nr_channels=64, channel_bw_MHz=300.0 / 64, nr_dms=64,
                  nr_samples=2000, nr_beams=2)
    plan, table, x, d_in = make_case(dd, s)
    d_out = out_buffer(s, fill=float("nan"))
    plan.execute(d_in, d_out, nr_beams=2)
    h_out = np.full((2, s.nr_dms, s.nr_samples), np.nan, dtype=np.float32)
    plan.execute_host(x, h_out, nr_beams=2)
    assert np.array_equal(h_out, d_out.cpu().numpy())
    plan.destroy()


def test_execute_host_async_pipeline_matches_oracle(dd):
    """dedisp_execute_host_async: seven batches through the three-slot pipeline (slots reused twice),
    every batch with its own pinned host buffers and its own data, bit-exact against the oracle."""
    import torch
    s = wl.scaled(wl.APERTIF, name="pipe", nr_channels=64, channel_bw_MHz=300.0 / 64, nr_dms=70,
                  nr_samples=1800, nr_beams=2, values="int16")
    plan = dd.Plan(*s.plan_args())
    table = oracle.shift_table(*s.table_args())
    h_ins, h_outs, refs = [], [], []
    for n in range(7):
        x = wl.make_input(wl.scaled(s, seed=1000 + 10 * n), plan.in_samples, plan.in_pitch)
        refs.append(oracle.dedisperse(x, table, s.nr_samples))
        h_ins.append(torch.from_numpy(x).pin_memory())
        h_outs.append(torch.full((s.nr_beams, s.nr_dms, s.nr_samples), -1.0).pin_memory())
    for h_in, h_out in zip(h_ins, h_outs):
        plan.execute_host_async(h_in, h_out, nr_beams=s.nr_beams)
    plan.host_sync()
    for n, (h_out, ref) in enumerate(zip(h_outs, refs)):
        assert np.array_equal(h_out.numpy().astype(np.float64), ref), "batch %d" % n
    # the synchronous entry point still works on the same plan afterwards, and sync is idempotent
    plan.execute_host(h_ins[0], h_outs[1], nr_beams=s.nr_beams)
    assert np.array_equal(h_outs[1].numpy().astype(np.float64), refs[0])
    plan.host_sync()
    plan.destroy()


@pytest.mark.parametrize("u8", [False, True])
def test_streaming_blocks_equal_one_long_dedispersion(dd, u8):
    """dedisp_stream_block_async over 6 consecutive blocks of a long series (the blocks share M input
    samples) equals the oracle run once on the whole series, bit-exactly."""
    import torch
    S, nblk = 1500, 6
    s = wl.scaled(wl.SURVEY8 if u8 else wl.APERTIF, name="stream", nr_channels=48,
                  channel_bw_MHz=300.0 / 48, nr_dms=61, nr_samples=S,
                  values="u8" if u8 else "int16", in_dtype=wl.U8 if u8 else wl.F32)
    plan = dd.Plan(*s.plan_args())
    table = oracle.shift_table(*s.table_args())
    M = plan.max_shift
    total = nblk * S
    long_setup = wl.scaled(s, nr_samples=total)
    series = wl.make_input(long_setup, total + M, total + M + 5)[0]   # [C][pitch], odd pitch
    ref = oracle.dedisperse(series[None], table, total)[0]
    h_series = torch.from_numpy(series).pin_memory()
    h_out = torch.full((s.nr_dms, total + 3), -1, dtype=torch.int32 if u8 else torch.float32).pin_memory()
    esz = 1 if u8 else 4
    for b in range(nblk):
        plan.stream_block_async(h_series, series.shape[1], h_out, total + 3, b * S)
        # the first block uploads S + M columns per row, every later one only its S new columns: the M
        # shared ones are carried over on the device
        assert plan.stream_h2d_bytes == s.nr_channels * (S + (M if b == 0 else 0)) * esz
    plan.host_sync()
    got = h_out.numpy()[:, :total]
    if u8:
        assert np.array_equal(got.view(np.uint32).astype(np.uint64), ref)
    else:
        assert np.array_equal(got.astype(np.float64), ref)
    assert (h_out.numpy()[:, total:] == -1).all()     # nothing written past the blocks
    # a block that does not continue the last one, and the block after a reset, upload everything; the
    # results are the same bits
    h_out.fill_(-1)
    for b, full in ((3, True), (4, False), (2, True), (3, False)):
        plan.stream_block_async(h_series, series.shape[1], h_out, total + 3, b * S)
        assert plan.stream_h2d_bytes == s.nr_channels * (S + (M if full else 0)) * esz
    plan.stream_reset()
    plan.stream_block_async(h_series, series.shape[1], h_out, total + 3, 4 * S)
    assert plan.stream_h2d_bytes == s.nr_channels * (S + M) * esz
    plan.host_sync()
    got = h_out.numpy()[:, 2 * S:5 * S]
    assert np.array_equal(got.view(np.uint32).astype(np.uint64) if u8 else got.astype(np.float64), ref[:, 2 * S:5 * S])
    with pytest.raises(dd.DedispError):
        plan.stream_block_async(h_series, series.shape[1], h_out, total + 3, total)  # past the end
    plan.destroy()


def test_streaming_with_shifts_longer_than_the_block_carries_them_over(dd):
    """The paper's LOFAR band at DM step 0.25: the max shift M is several times the block length
    S, so M of the S + M input columns of every block are already on the device.  8 consecutive blocks equal one
    long oracle run within the fp32 tolerance (Gaussian data), and every block after the first uploads
    nr_channels * S elements."""
    import torch
    S, nblk = 6000, 8
    s = wl.scaled(wl.LOFAR_PAPER, name="stream_long", nr_dms=64, nr_samples=S)
    plan = dd.Plan(*s.plan_args())
    table = oracle.shift_table(*s.table_args())
    M = plan.max_shift
    assert M >= 5 * S
    total = nblk * S
    series = wl.make_input(wl.scaled(s, nr_samples=total), total + M, total + M + 1)[0]
    ref, sabs = oracle.dedisperse(series[None], table, total, want_sabs=True)
    h_series = torch.from_numpy(series).pin_memory()
    h_out = torch.full((s.nr_dms, total), float("nan"), dtype=torch.float32).pin_memory()
    for b in range(nblk):
        plan.stream_block_async(h_series, series.shape[1], h_out, total, b * S)
        assert plan.stream_h2d_bytes == s.nr_channels * (S + (M if b == 0 else 0)) * 4
    plan.host_sync()
    err = np.abs(h_out.numpy().astype(np.float64) - ref[0])
    assert (err <= TOL * sabs[0]).all()
    plan.destroy()


def test_argument_errors_on_device(dd):
    import torch
    s = wl.TINY
    plan, table, x, d_in = make_case(dd, s)
    d_out = out_buffer(s)
    lib = dd.load_library()
    with pytest.raises(dd.DedispError) as e:
        plan.execute(d_in.data_ptr() + 4, d_out)   # misaligned base
    assert e.value.status == 1
    with pytest.raises(dd.DedispError):
        plan.execute(d_in, d_out, nr_beams=0)
    with pytest.raises(dd.DedispError):
        plan.execute(0, d_out)
    u8 = [v for v in range(dd.variant_count()) if dd.variant_name(v).startswith(("lds_u8", "generic_u8"))]
    assert u8 and not any(plan.variant_supported(v) for v in u8)
    with pytest.raises(dd.DedispError):
        plan.set_variant(u8[0])
    with pytest.raises(dd.DedispError):
        plan.execute_variant(u8[0], d_in, d_out)
    assert lib.dedisp_shift_table(plan._h, None) == 1
    # an oversized shift must be reported as OVERFLOW, not wrap
    with pytest.raises(dd.DedispError) as e:
        dd.Plan(4, 10.0, 0.1, 1e9, 16, 0.0, 1000.0, 64, wl.F32)
    assert e.value.status == 2
    plan.destroy()


def test_tuner_selects_persists_and_reloads(dd, tmp_path):
    s = wl.scaled(wl.APERTIF, name="tune", nr_channels=128, channel_bw_MHz=300.0 / 128,
                  nr_dms=256, nr_samples=4000)
    plan, table, x, d_in = make_case(dd, s)
    d_out = out_buffer(s)
    cache = str(tmp_path / "tune.tsv")
    ms = plan.tune(d_in, d_out, cache_path=cache)
    assert set(ms) == set(plan.supported_variants())
    best = min(ms, key=ms.get)
    assert plan.variant == best
    assert os.path.getsize(cache) > 0
    # the tuned plan still computes the right thing
    ref, sabs = oracle.dedisperse(x, table, s.nr_samples, want_sabs=True)
    d_out.fill_(float("nan"))
    plan.execute(d_in, d_out)
    check_full(s, to_host(s, d_out), ref, sabs, False)
    # a fresh plan picks the winner up from the cache; another setup is left alone
    with dd.Plan(*s.plan_args()) as p2:
        p2.set_variant(0)
        assert p2.load_tuning(cache) is True
        assert p2.variant == best
    with dd.Plan(*wl.TINY.plan_args()) as p3:
        before = p3.variant
        assert p3.load_tuning(cache) is False
        assert p3.variant == before
    # the key carries a batch-size class (1 / 2-7 / >= 8 beams): a 40-beam winner does not overwrite the
    # single-beam one; a class without an entry falls back to one that has
    other = [v for v in plan.supported_variants() if v != best][0]
    line = open(cache).read().splitlines()[-1]
    assert ";beams=1\t" in line
    with open(cache, "a") as f:
        f.write(line.replace(";beams=1\t", ";beams=8\t").replace(dd.variant_name(best), dd.variant_name(other)) + "\n")
    with dd.Plan(*s.plan_args()) as p4:
        assert p4.load_tuning(cache, nr_beams=40) and p4.variant == other
        assert p4.load_tuning(cache, nr_beams=1) and p4.variant == best
        assert p4.load_tuning(cache, nr_beams=3) and p4.variant in (best, other)
    with pytest.raises(dd.DedispError) as e:
        plan.load_tuning(str(tmp_path / "missing.tsv"))
    assert e.value.status == 5
    plan.destroy()
