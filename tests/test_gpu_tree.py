"""KIND_TREE kernels (kernel_tree.cuh): which plans get them, and parity where the slope classes,
the ragged DM groups and the staging ring are stressed."""
import numpy as np
import pytest

import oracle
from paper_1601_01165_b200 import workloads as wl
from test_gpu_parity import check_full, dd, make_case, out_buffer, to_host  # noqa: F401

pytestmark = pytest.mark.gpu


def tree_variants(dd, plan):
    return [v for v in plan.supported_variants() if dd.variant_name(v).startswith("tree_")]


def max_q(table):
    """largest per-channel minimum increment (the q_c of DESIGN.md section 5), from the oracle table"""
    if table.shape[0] < 2:
        return 0
    return int(np.diff(table.astype(np.int64), axis=0).min(axis=0).max())


@pytest.mark.parametrize("name,expect", [("tiny", True), ("apertif", True), ("survey8", True),
                                         ("batch40", True), ("lofar", False)])
def test_which_configs_get_tree_kernels(dd, name, expect):
    s = wl.CONFIGS[name]
    with dd.Plan(*s.plan_args()) as plan:
        tv = tree_variants(dd, plan)
        assert bool(tv) == expect
        table = oracle.shift_table(*s.table_args())
        inc = np.diff(table.astype(np.int64), axis=0)
        ok = bool(((inc.max(axis=0) - inc.min(axis=0)) <= 1).all())
        assert ok  # every BASELINE table is a rounded linear function of the DM index
        for v in tv:  # a variant is only offered when its lattice covers the plan's slope classes
            qcap = int(dd.variant_name(v).split(" q")[1].split()[0])
            assert qcap >= max_q(table)
        if name == "lofar":
            assert max_q(table) > 7


def run_tree(dd, setup, exact):
    plan, table, x, d_in = make_case(dd, setup)
    ref, sabs = oracle.dedisperse(x, table, setup.nr_samples, want_sabs=True)
    tv = tree_variants(dd, plan)
    for v in tv:
        d_out = out_buffer(setup, fill=-1 if setup.in_dtype == wl.U8 else float("nan"))
        plan.execute_variant(v, d_in, d_out, nr_beams=setup.nr_beams)
        try:
            check_full(setup, to_host(setup, d_out), ref, sabs, exact)
        except AssertionError as e:
            raise AssertionError("%s on %s: %s" % (dd.variant_name(v), setup.name, e))
    plan.destroy()
    return len(tv), max_q(table)


def test_slope_class_4_only_runs_q4_lattices(dd):
    # survey8 band, lowest channels: q_c reaches 4; integer data -> bit-exact
    s = wl.scaled(wl.SURVEY8, name="q4_f32", nr_channels=96, channel_bw_MHz=300.0 / 96, nr_dms=131,
                  nr_samples=2900, in_dtype=wl.F32, values="int16")
    n, q = run_tree(dd, s, exact=True)
    assert q == 4 and n >= 3
    s8 = wl.scaled(wl.SURVEY8, name="q4_u8", nr_channels=96, channel_bw_MHz=300.0 / 96, nr_dms=131,
                   nr_samples=2900)
    n, q = run_tree(dd, s8, exact=True)
    assert q == 4 and n >= 3


def test_slope_classes_up_to_7_run_the_coarse_grid_lattices(dd):
    # Apertif band with a DM step of 0.5: shifts grow by up to 6.6 samples per step at the lowest channel
    s = wl.scaled(wl.APERTIF, name="q6_f32", nr_channels=96, channel_bw_MHz=300.0 / 96, nr_dms=101,
                  nr_samples=2700, dm_step=0.5, values="int16")
    n, q = run_tree(dd, s, exact=True)
    assert q == 6 and n >= 2
    s8 = wl.scaled(s, name="q6_u8", in_dtype=wl.U8, values="u8")
    n, q = run_tree(dd, s8, exact=True)
    assert q == 6 and n >= 1


def test_slope_beyond_the_lattice_falls_back_to_other_kinds(dd):
    s = wl.scaled(wl.SURVEY8, name="q9", nr_channels=64, channel_bw_MHz=300.0 / 64, nr_dms=40,
                  nr_samples=1500, dm_step=0.5, in_dtype=wl.F32, values="int16")
    with dd.Plan(*s.plan_args()) as plan:
        assert max_q(oracle.shift_table(*s.table_args())) > 7
        assert not tree_variants(dd, plan)
        assert plan.supported_variants()  # lds / generic still run it


def test_many_chunks_ragged_everything_bit_exact(dd):
    # 37 chunks of 8 channels + a ragged one, DMs not a multiple of 4/6/8, samples not a tile multiple
    s = wl.scaled(wl.APERTIF, name="ring", nr_channels=301, channel_bw_MHz=300.0 / 301, nr_dms=157,
                  nr_samples=2051, values="int16")
    n, _ = run_tree(dd, s, exact=True)
    assert n >= 8
    s8 = wl.scaled(wl.SURVEY8, name="ring_u8", nr_channels=301, channel_bw_MHz=300.0 / 301,
                   nr_dms=157, nr_samples=2064)
    n, _ = run_tree(dd, s8, exact=True)
    assert n >= 3


def test_shipped_winner_for_apertif_is_a_tree_kernel(dd):
    from paper_1601_01165_b200 import tuning
    with dd.Plan(*wl.APERTIF.plan_args()) as plan:
        tuning.apply_shipped(plan)
        assert dd.variant_name(plan.variant).startswith("tree_f32")


@pytest.mark.parametrize("name,kind", [("apertif", "tree_f32"), ("survey8", "tree_u8"),
                                       ("lofar", "lds_f32"), ("batch40", "tree_f32")])
def test_untuned_default_picks_the_right_kernel_family(dd, name, kind):
    """Without a tuning cache the plan's cost model must land in the family the tuner picks
    (DESIGN.md section 8)."""
    with dd.Plan(*wl.CONFIGS[name].plan_args()) as plan:
        assert dd.variant_name(plan.variant).startswith(kind)
        assert plan.variant_supported(plan.variant)


def test_long_shift_setup_uses_a_staged_kernel(dd):
    """The paper's LOFAR setup (DM step 0.25: hundreds of samples per DM step): tree kernels are out,
    the long-span lds variants fit; every supported variant stays exact."""
    s = wl.Setup("lofar_paper_s", 32, 138.0, 6.0 / 32, 200000.0, 9000, 0.0, 0.25, 24, values="int16",
                 seed=77)
    plan, table, x, d_in = make_case(dd, s)
    assert not tree_variants(dd, plan)
    names = [dd.variant_name(v) for v in plan.supported_variants()]
    assert any(n.startswith("lds_f32: 4x2048") or n.startswith("lds_f32: 4x4096") for n in names)
    ref = oracle.dedisperse(x, table, s.nr_samples)
    ran = 0
    for v in plan.supported_variants():
        d_out = out_buffer(s, fill=-1.0)
        plan.execute_variant(v, d_in, d_out)
        assert np.array_equal(to_host(s, d_out).astype(np.float64), ref), dd.variant_name(v)
        ran += 1
    assert ran >= 3
    plan.destroy()


@pytest.mark.parametrize("base", ["apertif", "survey8"])
def test_lazy_window_twins_are_bit_identical(dd, base):
    """A LAZY lattice loads the same words later, it does not change a single add or its order: on Gaussian
    fp32 data (where the tolerance against the oracle would hide a changed order) every lazy variant must
    reproduce its up-front twin bit for bit; likewise on uint8."""
    import torch
    s = wl.scaled(wl.CONFIGS[base], name=base + "_twins", nr_dms=333, nr_samples=3001)
    plan, table, x, d_in = make_case(dd, s)
    names = {dd.variant_name(v): v for v in tree_variants(dd, plan)}
    pairs = [(v, names[n[:-len(" lazy")]]) for n, v in names.items()
             if n.endswith(" lazy") and n[:-len(" lazy")] in names]
    assert len(pairs) >= 4
    for lazy, plain in pairs:
        a = out_buffer(s, fill=-1 if s.in_dtype == wl.U8 else float("nan"))
        b = out_buffer(s, fill=-2 if s.in_dtype == wl.U8 else float("nan"))
        plan.execute_variant(lazy, d_in, a, nr_beams=s.nr_beams)
        plan.execute_variant(plain, d_in, b, nr_beams=s.nr_beams)
        assert torch.equal(a.view(torch.int32), b.view(torch.int32)), dd.variant_name(lazy)
    plan.destroy()


def test_persistent_ctas_cross_tiles_and_beams_on_every_fp32_variant(dd):
    """The fp32 tree kernels run as persistent CTAs whose chunk ring runs on across tiles.  The scaled
    configs of the other tests have fewer tiles than the GPU has SMs; here every compiled fp32 tree tile
    gets more than 2 x 148 tiles over two beams (so every CTA crosses tile and beam boundaries), with a
    channel count that leaves a ragged last chunk for every stage depth (70 = 3 x 20 + 10 = 4 x 16 + 6 =
    5 x 12 + 10 = 8 x 8 + 6), ragged DM and time tiles, integer-valued data: exact."""
    s = wl.scaled(wl.APERTIF, name="persist", nr_channels=70, channel_bw_MHz=300.0 / 70, nr_dms=700,
                  nr_samples=9001, nr_beams=2, values="int16")
    n, q = run_tree(dd, s, exact=True)
    assert n >= 30 and q >= 3
