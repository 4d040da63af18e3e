"""dedisp_execute_static_scratch: the uint8 path for callers that cannot allocate device memory.

Some users of this library run where cudaMalloc is not an option: inside a process whose free device
memory already belongs to a pool allocator (a raw cudaMalloc then reports out-of-memory although the
pool has room), inside a real-time block loop (cudaMalloc / cudaFree serialise the device and stall
the other beams' streams), or beside a thread that captures a CUDA graph in the global capture mode
(an allocation call is refused there and breaks the capture).  For them the library keeps the uint8
kernels' pair scratch in a fixed 16 MiB array inside the library image instead of the plan's
cudaMalloc'ed workspace (include/dedisp.h, csrc/static_scratch.cu).

The array is shared by every call and keeps the previous call's contents, so the checks below run
calls back to back that differ in plan, row length and data: each result must be bit-identical to
dedisp_execute on the same plan (the tolerance of every uint8 test in this suite: exact) and to the
oracle.  This file is collected last on purpose (`pytest --collect-only`): the array outlives every
test, and a failure here under `pytest -x` then hides nothing after it.  Nothing else in the suite
touches the array, so the tests pass alone in a fresh process and after the rest of the suite.
"""
import numpy as np
import pytest

import oracle
from paper_1601_01165_b200 import workloads as wl
from test_gpu_parity import dd, make_case, out_buffer, to_host  # noqa: F401

pytestmark = pytest.mark.gpu


def scratch_need_bytes(plan):
    """include/dedisp.h: one beam needs nr_channels * PAIR_PITCH * 4 bytes."""
    s2 = ((plan.nr_samples + 1) // 2 + 3) & ~3
    pair_pitch = (s2 + plan.max_shift + 3) & ~3
    assert pair_pitch == plan.pair_pitch
    return plan.nr_channels * pair_pitch * 4


def tree_u8_case(dd, setup):
    plan, table, x, d_in = make_case(dd, setup)
    tree = [v for v in plan.supported_variants() if dd.variant_name(v).startswith("tree_u8")]
    assert tree, "no tree_u8 variant supports %s" % setup.name
    plan.set_variant(tree[0])
    return plan, table, x, d_in


def run_both(dd, setup, plan, d_in, stream=None):
    """The existing path and the static-scratch path on the same plan and input, poisoned outputs."""
    import torch
    want = out_buffer(setup, fill=-1)
    plan.execute(d_in, want, nr_beams=setup.nr_beams)
    torch.cuda.synchronize()
    got = out_buffer(setup, fill=-1)
    plan.execute_static_scratch(d_in, got, nr_beams=setup.nr_beams, stream=stream)
    torch.cuda.synchronize()
    return got, want


BIG = wl.Setup("static_a", 300, 1220.0, 300.0 / 300, 24414.0, 4100, 0.0, 0.2, 150, nr_beams=2,
               in_dtype=wl.U8, values="u8", seed=31)
# shorter rows, fewer channels, odd S: the scratch still holds BIG's pairs past and between these rows
SMALL = wl.Setup("static_b", 37, 1400.0, 3.0, 20000.0, 1021, 0.0, 0.25, 45, in_dtype=wl.U8, values="u8",
                 seed=32)


def test_two_calls_in_a_row_match_the_existing_path_and_the_oracle(dd):
    import torch
    assert dd.static_scratch_bytes() == 16 << 20
    pa, ta, xa, da = tree_u8_case(dd, BIG)
    pb, tb, xb, db = tree_u8_case(dd, SMALL)
    assert scratch_need_bytes(pa) <= dd.static_scratch_bytes()
    st = torch.cuda.Stream()
    # call 1 (the first on this device also looks the array's address up), then call 2 on another plan with
    # other data and a smaller footprint, then plan A again with the rows reversed: whatever a call leaves
    # in the array must not reach the next one's result
    for setup, plan, x, table, d_in, stream in ((BIG, pa, xa, ta, da, None), (SMALL, pb, xb, tb, db, st),
                                                (BIG, pa, xa[:, ::-1].copy(), ta, None, None)):
        if d_in is None:
            d_in = torch.from_numpy(x).cuda()
        got, want = run_both(dd, setup, plan, d_in, stream)
        assert torch.equal(got, want), setup.name
        ref = oracle.dedisperse(x, table, setup.nr_samples)
        assert np.array_equal(to_host(setup, got).astype(np.uint64), ref), setup.name
    # a repeat of the last call leaves the amount of free device memory as it was: nothing was allocated
    free0 = torch.cuda.mem_get_info()[0]
    got2 = out_buffer(BIG, fill=-1)
    free1 = torch.cuda.mem_get_info()[0]          # after the test's own output buffer
    pa.execute_static_scratch(d_in, got2, nr_beams=BIG.nr_beams)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free1 <= free0
    assert torch.equal(got2, got)
    pa.destroy()
    pb.destroy()


def test_a_batch_larger_than_the_array_goes_through_it_in_groups(dd):
    """3 beams of 5.9 MiB of pairs each: two fit the 16 MiB array, so the call runs two groups in stream order."""
    import torch
    s = wl.Setup("static_groups", 512, 1220.0, 300.0 / 512, 24414.0, 5600, 0.0, 0.2, 40, nr_beams=3,
                 in_dtype=wl.U8, values="u8", seed=33)
    plan, table, x, d_in = tree_u8_case(dd, s)
    need = scratch_need_bytes(plan)
    assert need <= dd.static_scratch_bytes() < 3 * need
    got, want = run_both(dd, s, plan, d_in)
    assert torch.equal(got, want)
    assert np.array_equal(to_host(s, got).astype(np.uint64), oracle.dedisperse(x, table, s.nr_samples))
    plan.destroy()


def test_sizes_beyond_the_array_and_plans_without_scratch_are_refused(dd):
    import torch
    # survey-length rows: 1536 channels x ~24.6k pairs x 4 B = 151 MB of scratch per beam
    s = wl.scaled(wl.SURVEY8, name="static_too_big", nr_dms=8)
    with dd.Plan(*s.plan_args()) as plan:
        tree = [v for v in plan.supported_variants() if dd.variant_name(v).startswith("tree_u8")]
        plan.set_variant(tree[0])
        assert scratch_need_bytes(plan) > dd.static_scratch_bytes()
        d_in = torch.zeros((1, s.nr_channels, plan.in_pitch), dtype=torch.uint8, device="cuda")
        d_out = out_buffer(s, fill=-1)
        with pytest.raises(dd.DedispError) as e:
            plan.execute_static_scratch(d_in, d_out)
        assert e.value.status == 1                                    # DEDISP_ERR_INVALID_ARG
        assert str(scratch_need_bytes(plan)) in str(e.value) and str(16 << 20) in str(e.value)
        torch.cuda.synchronize()
        assert (d_out == -1).all()                                    # nothing was launched
        plan.execute(d_in, d_out)                                     # the allocating path still serves it
        torch.cuda.synchronize()
        assert (d_out == 0).all()
    # fp32 plans, and uint8 plans on a kernel that reads the input directly, use no scratch memory
    with dd.Plan(*wl.TINY.plan_args()) as f32:
        d_in = torch.zeros((1, wl.TINY.nr_channels, f32.in_pitch), dtype=torch.float32, device="cuda")
        with pytest.raises(dd.DedispError) as e:
            f32.execute_static_scratch(d_in, out_buffer(wl.TINY))
        assert e.value.status == 1 and "dedisp_execute" in str(e.value)
    with dd.Plan(*SMALL.plan_args()) as u8:
        lds = [v for v in u8.supported_variants() if dd.variant_name(v).startswith("lds_u8")]
        u8.set_variant(lds[0])
        d_in = torch.zeros((1, SMALL.nr_channels, u8.in_pitch), dtype=torch.uint8, device="cuda")
        with pytest.raises(dd.DedispError) as e:
            u8.execute_static_scratch(d_in, out_buffer(SMALL))
        assert e.value.status == 1
