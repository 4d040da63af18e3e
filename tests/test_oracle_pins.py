"""Pins for the CPU oracle (oracle/dedisp_oracle.c) against what the paper and the
mathematics fix -- NOT against itself and never against the CUDA path.

Each test says which plausible mistake it would catch.
"""
import json
import os
from fractions import Fraction

import numpy as np
import pytest

import oracle
from paper_1601_01165_b200 import workloads as wl

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")
with open(os.path.join(GOLDEN, "shift_table_survey.json")) as f:
    SURVEY = json.load(f)
with open(os.path.join(GOLDEN, "paper_constants.json")) as f:
    PAPER = json.load(f)

TABLE_SETUPS = [wl.TINY, wl.APERTIF, wl.LOFAR, wl.SURVEY8]
_tables = {}


def table(setup):
    if setup.name not in _tables:
        _tables[setup.name] = oracle.shift_table(*setup.table_args())
    return _tables[setup.name]


# ---------------------------------------------------------------- Eq. (1) ----

def test_delay_closed_form_literals():
    """Eq. (1) with f_h -> infinity is k = 4150*DM/f^2 seconds.
    Literals worked by hand: catches a wrong constant, f instead of f^2, MHz/Hz
    mix-ups, or DM entering non-linearly."""
    inf = 1e150
    assert oracle.delay_samples(1000.0, inf, 1.0, 1.0) == pytest.approx(4.150e-3, rel=1e-15)
    assert oracle.delay_samples(2000.0, inf, 1.0, 1.0) == pytest.approx(1.0375e-3, rel=1e-15)
    assert oracle.delay_samples(1000.0, inf, 3.0, 1.0) == pytest.approx(12.45e-3, rel=1e-15)
    # times the sample rate (north star): 20 kHz
    assert oracle.delay_samples(1000.0, inf, 1.0, 20000.0) == pytest.approx(83.0, rel=1e-15)
    assert PAPER["dispersion_constant"]["value"] == 4150.0


def test_delay_sign_and_reference_frequency():
    """'the highest frequency f_h is received at t_x, lower ones at t_x + k'
    (PAPER.md:34): zero at f_h, positive below it, negative above it.  Catches a
    swapped (1/f_h^2 - 1/f^2)."""
    for dm in (0.0, 0.25, 17.0, 511.75):
        assert oracle.delay_samples(1720.0, 1720.0, dm, 20000.0) == 0.0
        assert oracle.shift_of(1720.0, 1720.0, dm, 20000.0) == 0
    assert oracle.delay_samples(1420.0, 1720.0, 10.0, 20000.0) > 0
    assert oracle.delay_samples(1800.0, 1720.0, 10.0, 20000.0) < 0
    # hand value, tiny config: c=0 (1420 MHz), f_h = 1452, DM 127, 1 kHz:
    # 4150*127*(1/1420^2 - 1/1452^2)*1000 = 11.39 -> 11
    x = oracle.delay_samples(1420.0, 1452.0, 127.0, 1000.0)
    assert 11.38 < x < 11.40
    assert oracle.round_half_up(x) == 11


def test_round_half_up_rule():
    """Reading A4: nearest, ties up (all operands exact)."""
    for x, r in [(0.0, 0), (0.49999999999999994, 0), (0.5, 1), (1.5, 2), (2.5, 3),
                 (10499.5, 10500), (31498.5, 31499), (7.000000001, 7), (6.999999999, 7)]:
        assert oracle.round_half_up(x) == r


def test_f_high_reading_a1_reproduces_baseline_padding():
    """BASELINE.json states the max shifts (~6.7k, ~73k, ~19.8k).  Only the
    band-top reading f_h = f_low + C*bw gives them; f_h = top channel gives
    70659 for LOFAR, outside the tolerance.  Catches the wrong f_h or channel
    labelling (f_c must be f_low + c*bw with c = 0 the lowest)."""
    for name in ("apertif", "lofar", "survey8"):
        s = wl.CONFIGS[name]
        M = int(table(s).max())
        p = SURVEY["padding"][name]
        assert abs(M - p["approx"]) <= p["tol"], (name, M)
    s = wl.LOFAR
    assert oracle.f_high_MHz(s.f_low_MHz, s.channel_bw_MHz, s.nr_channels) == 144.0
    assert oracle.channel_freq_MHz(s.f_low_MHz, s.channel_bw_MHz, 0) == 138.0
    assert oracle.channel_freq_MHz(s.f_low_MHz, s.channel_bw_MHz, 16) == 141.0


@pytest.mark.parametrize("setup", TABLE_SETUPS, ids=lambda s: s.name)
def test_table_structure(setup):
    """Properties Eq. (1) forces on the table: zero row at DM 0, non-negative,
    non-decreasing in DM, non-increasing in channel (higher f -> smaller delay),
    maximum at (last DM, channel 0).  Catches transposed [C][D] output and a
    reversed channel order."""
    t = table(setup)
    assert t.shape == (setup.nr_dms, setup.nr_channels) and t.dtype == np.int32
    assert (t[0] == 0).all()                       # dm_first = 0
    assert (t >= 0).all()
    assert (np.diff(t.astype(np.int64), axis=0) >= 0).all()
    assert (np.diff(t.astype(np.int64), axis=1) <= 0).all()
    assert t.max() == t[-1, 0]
    assert t[-1, 0] > t[-1, -1]


@pytest.mark.parametrize("setup", TABLE_SETUPS, ids=lambda s: s.name)
def test_table_matches_survey_prototype(setup):
    """Independent NumPy prototype of the survey: max, sum of all
    entries and three spot entries."""
    t = table(setup).astype(np.int64)
    g = SURVEY["survey"][setup.name]
    C, D = setup.nr_channels, setup.nr_dms
    assert int(t.max()) == g["max_shift"]
    assert int(t.sum()) == g["sum"]
    assert int(t[D - 1, C // 2]) == g["mid_last"]
    assert int(t[D - 1, C - 1]) == g["top_last"]
    assert int(t[1, 0]) == g["c0_dm1"]


def _exact_delay(setup, i, c):
    """Eq. (1) x rate in exact rational arithmetic on the double-valued dm_i, f_c, f_h."""
    dm = Fraction(oracle.trial_dm(setup.dm_first, setup.dm_step, i))
    f = Fraction(oracle.channel_freq_MHz(setup.f_low_MHz, setup.channel_bw_MHz, c))
    fh = Fraction(oracle.f_high_MHz(setup.f_low_MHz, setup.channel_bw_MHz, setup.nr_channels))
    return 4150 * dm * (1 / (f * f) - 1 / (fh * fh)) * Fraction(setup.sample_rate)


@pytest.mark.parametrize("setup", TABLE_SETUPS, ids=lambda s: s.name)
def test_table_against_exact_rational_arithmetic(setup):
    """A different arithmetic (exact fractions) on a lattice of entries: the table
    entry must be round-half-up of the exact value wherever the exact value is
    not within 1e-6 of a tie.  Catches dropped terms, wrong association that
    loses precision, float32 intermediates, truncation instead of rounding."""
    t = table(setup)
    D, C = t.shape
    ii = sorted(set(list(range(0, D, max(1, D // 61))) + [1, D - 1]))
    cc = sorted(set(list(range(0, C, max(1, C // 29))) + [C - 1]))
    near_ties = 0
    for i in ii:
        for c in cc:
            x = _exact_delay(setup, i, c)
            fl = x.numerator // x.denominator
            frac = x - fl
            if abs(frac - Fraction(1, 2)) < Fraction(1, 10 ** 6):
                near_ties += 1
                assert int(t[i, c]) in (fl, fl + 1)
                continue
            assert int(t[i, c]) == fl + (1 if frac >= Fraction(1, 2) else 0), (i, c)
            # the double itself is accurate to a few ulp
            xd = oracle.delay_samples(float(oracle.channel_freq_MHz(setup.f_low_MHz, setup.channel_bw_MHz, c)),
                                      oracle.f_high_MHz(setup.f_low_MHz, setup.channel_bw_MHz, C),
                                      oracle.trial_dm(setup.dm_first, setup.dm_step, i), setup.sample_rate)
            # a - b cancels near the top of the band, so the error bound is relative
            # to the un-cancelled magnitude 4150*dm*rate/f_c^2 (a few ulp of it)
            mag = 4150 * Fraction(oracle.trial_dm(setup.dm_first, setup.dm_step, i)) \
                * Fraction(setup.sample_rate) / Fraction(oracle.channel_freq_MHz(
                    setup.f_low_MHz, setup.channel_bw_MHz, c)) ** 2
            assert abs(Fraction(xd) - x) <= 8 * mag / 2 ** 53
    assert near_ties <= 4


def test_lofar_half_integer_ties_follow_canonical_association():
    """Reading A3: the LOFAR-like table has mathematically half-integer entries;
    the canonical association ((4150*dm)*diff)*rate decides them.  Values from
    the survey's NumPy prototype (not paper-printed)."""
    s = wl.LOFAR
    t = table(s)
    fh = oracle.f_high_MHz(s.f_low_MHz, s.channel_bw_MHz, s.nr_channels)
    for e in SURVEY["lofar_ties"]["entries"]:
        i, c = e["dm_index"], e["channel"]
        x = oracle.delay_samples(oracle.channel_freq_MHz(s.f_low_MHz, s.channel_bw_MHz, c), fh,
                                 oracle.trial_dm(s.dm_first, s.dm_step, i), s.sample_rate)
        assert x == float.fromhex(e["x_hex"])
        assert int(t[i, c]) == e["shift"]
        # and the exact value really is (within 1e-9 of) a tie
        assert abs(_exact_delay(s, i, c) % 1 - Fraction(1, 2)) < Fraction(1, 10 ** 9)


def test_trial_dm_is_computed_not_accumulated():
    """Reading A5: dm_i = dm_first + i*dm_step in double (0.01 is inexact)."""
    assert oracle.trial_dm(0.0, 0.01, 1620) == 16.2
    acc = 0.0
    for _ in range(1620):
        acc += 0.01
    assert acc != 16.2 and oracle.trial_dm(0.0, 0.01, 1620) != acc
    assert oracle.trial_dm(1.5, 0.25, 8) == 3.5


# ------------------------------------------------------------ Algorithm 1 ----

def _gather_reference(x, shift, S):
    """Second, index-arithmetic-free restatement: NumPy fancy-indexing gather."""
    x = x if x.ndim == 3 else x[None]
    B, C, _ = x.shape
    D = shift.shape[0]
    t_idx = np.arange(S)[None, None, :] + shift.astype(np.int64)[:, :, None]     # [D][C][S]
    c_idx = np.arange(C)[None, :, None]
    acc_t = np.uint64 if x.dtype == np.uint8 else np.float64
    return np.stack([x[b][c_idx, t_idx].astype(acc_t).sum(axis=1) for b in range(B)])


def _rand_table(rng, D, C, smax):
    return rng.integers(0, smax + 1, size=(D, C)).astype(np.int32)


def test_dm0_row_is_plain_channel_sum():
    """'every output element is the sum of c samples: one for each frequency
    channel': with zero shifts the row is numpy's channel sum."""
    rng = np.random.default_rng(1)
    C, S, M = 13, 200, 7
    x = rng.integers(0, 16, size=(C, S + M)).astype(np.float32)
    shift = np.zeros((3, C), dtype=np.int32)
    out = oracle.dedisperse(x, shift, S)
    assert out.shape == (1, 3, S)
    for i in range(3):
        assert np.array_equal(out[0, i], x[:, :S].astype(np.float64).sum(axis=0))
    # on the real tiny table, row 0 is the DM-0 trial
    t = table(wl.TINY)
    xin = wl.make_input(wl.TINY, 1024 + 11, 1036, pulse_shifts=t[64])
    out = oracle.dedisperse(xin, t, 1024)
    assert np.array_equal(out[0, 0], xin[0, :, :1024].astype(np.float64).sum(axis=0))


def test_constant_input_gives_channel_count():
    rng = np.random.default_rng(2)
    C, D, S, M = 9, 5, 64, 12
    shift = _rand_table(rng, D, C, M)
    x = np.ones((C, S + M), dtype=np.float32)
    assert (oracle.dedisperse(x, shift, S) == C).all()
    xb = np.full((C, S + M), 3, dtype=np.uint8)
    assert (oracle.dedisperse(xb, shift, S) == 3 * C).all()


def test_single_channel_is_a_pure_shift():
    """Only channel c0 non-zero -> out[i][t] = in[c0][t + shift[i][c0]]: catches
    shift[c][dm] vs shift[dm][c] transposition and a '-' instead of '+' in the
    index (reading A10, Alg. 1 line 'sample + Delta')."""
    rng = np.random.default_rng(3)
    C, D, S, M = 6, 7, 50, 20
    shift = _rand_table(rng, D, C, M)
    for c0 in (0, 2, 5):
        x = np.zeros((C, S + M), dtype=np.float32)
        x[c0] = rng.integers(1, 100, size=S + M)
        out = oracle.dedisperse(x, shift, S)[0]
        for i in range(D):
            assert np.array_equal(out[i], x[c0, shift[i, c0]:shift[i, c0] + S].astype(np.float64))


@pytest.mark.parametrize("dtype", [np.float32, np.uint8])
def test_brute_force_gather_random_tables(dtype):
    """Tiny random shapes against the fancy-indexing gather, arbitrary (even
    non-monotone) tables, several beams, pitch > S+M."""
    rng = np.random.default_rng(4)
    for (B, C, D, S, M, pad) in [(1, 1, 1, 1, 0, 0), (2, 3, 4, 17, 5, 3), (3, 8, 8, 64, 31, 0),
                                 (1, 5, 2, 33, 100, 7)]:
        shift = _rand_table(rng, D, C, M)
        if dtype == np.uint8:
            x = rng.integers(0, 256, size=(B, C, S + M + pad), dtype=np.uint8)
        else:
            x = rng.integers(-50, 50, size=(B, C, S + M + pad)).astype(np.float32)
        out = oracle.dedisperse(x, shift, S)
        assert out.dtype == (np.uint64 if dtype == np.uint8 else np.float64)
        assert np.array_equal(out, _gather_reference(x, shift, S))


def test_linearity_on_integer_data():
    rng = np.random.default_rng(5)
    C, D, S, M = 7, 6, 40, 9
    shift = _rand_table(rng, D, C, M)
    x = rng.integers(0, 16, size=(C, S + M)).astype(np.float32)
    y = rng.integers(0, 16, size=(C, S + M)).astype(np.float32)
    lhs = oracle.dedisperse(3 * x + 2 * y, shift, S)
    assert np.array_equal(lhs, 3 * oracle.dedisperse(x, shift, S) + 2 * oracle.dedisperse(y, shift, S))


def test_beams_are_independent():
    """every beam can be processed independently."""
    rng = np.random.default_rng(6)
    B, C, D, S, M = 4, 5, 6, 30, 8
    shift = _rand_table(rng, D, C, M)
    x = rng.standard_normal((B, C, S + M)).astype(np.float32)
    out, sabs = oracle.dedisperse(x, shift, S, want_sabs=True)
    for b in range(B):
        o1, s1 = oracle.dedisperse(x[b], shift, S, want_sabs=True)
        assert np.array_equal(out[b], o1[0]) and np.array_equal(sabs[b], s1[0])
    assert np.allclose(sabs, _gather_reference(np.abs(x), shift, S), rtol=1e-14)


def test_injected_pulse_peaks_at_its_dm_and_time():
    """BASELINE config 1: amplitude-100 pulse dispersed at DM index 64 arriving at
    t = 300 must be the unique maximum at exactly (64, 300), and exceed the noise
    sum there by C*100 = 3200 (readings A13/A14)."""
    s = wl.TINY
    t = table(s)
    M = int(t.max())
    pitch = 1036
    x = wl.make_input(s, s.nr_samples + M, pitch, pulse_shifts=t[64])
    noise = wl.make_input(wl.scaled(s, pulse=None), s.nr_samples + M, pitch)
    valid = x[..., :s.nr_samples + M]           # the pitch padding is poisoned and never read
    assert valid.max() <= 115 and np.array_equal(valid, np.round(valid))
    assert np.isnan(x[..., s.nr_samples + M:]).all()
    out = oracle.dedisperse(x, t, s.nr_samples)[0]
    assert np.unravel_index(np.argmax(out), out.shape) == (64, 300)
    assert (out == out.max()).sum() == 1
    base = oracle.dedisperse(noise, t, s.nr_samples)[0]
    assert out[64, 300] - base[64, 300] == 3200.0
    # duplicate table rows (110 of 128 are distinct) give identical output rows
    rows = {}
    for i in range(s.nr_dms):
        rows.setdefault(t[i].tobytes(), []).append(i)
    assert len(rows) == 110
    for idx in rows.values():
        for i in idx[1:]:
            assert np.array_equal(out[i], out[idx[0]])


@pytest.mark.parametrize("dtype", [np.float32, np.uint8])
def test_points_variant_equals_full(dtype):
    rng = np.random.default_rng(7)
    B, C, D, S, M = 3, 11, 9, 70, 25
    shift = _rand_table(rng, D, C, M)
    if dtype == np.uint8:
        x = rng.integers(0, 256, size=(B, C, S + M), dtype=np.uint8)
    else:
        x = rng.standard_normal((B, C, S + M)).astype(np.float32)
    full, sabs = oracle.dedisperse(x, shift, S, want_sabs=True)
    pts = np.stack([rng.integers(0, B, 200), rng.integers(0, D, 200), rng.integers(0, S, 200)], 1)
    got, gs = oracle.dedisperse_points(x, shift, S, pts, want_sabs=True)
    assert np.array_equal(got, full[pts[:, 0], pts[:, 1], pts[:, 2]])
    if dtype == np.float32:
        assert np.array_equal(gs, sabs[pts[:, 0], pts[:, 1], pts[:, 2]])
    assert np.array_equal(got, _gather_reference(x, shift, S)[pts[:, 0], pts[:, 1], pts[:, 2]])


def test_reads_outside_row_are_rejected():
    x = np.zeros((2, 10), dtype=np.float32)
    with pytest.raises(AssertionError):
        oracle.dedisperse(x, np.array([[0, 3]], dtype=np.int32), 8)


# ------------------------------------------------- metric conventions (paper) --

def test_flop_convention_matches_paper():
    """One flop per (dm, sample, channel): PAPER.md:105 and :193."""
    assert wl.APERTIF.adds_per_beam // wl.APERTIF.nr_dms == 20000 * 1024
    assert round(wl.APERTIF.adds_per_beam / wl.APERTIF.nr_dms / 1e6) == round(20.48)
    assert abs(wl.APERTIF.adds_per_beam / wl.APERTIF.nr_dms / 1e6 - PAPER["mflop_per_dm"]["apertif"]["value"]) < 0.5
    assert abs(wl.LOFAR.adds_per_beam / wl.LOFAR.nr_dms / 1e6 - PAPER["mflop_per_dm"]["lofar"]["value"]) < 0.5
    inst = PAPER["apertif_instrument"]
    tf = inst["beams"] * inst["dms"] * 20000 * 1024 / 1e12     # per second of data
    assert abs(tf - inst["tflops"]) < 0.1
    r = PAPER["apertif_data_rates_GBps"]
    assert abs(450 * 1024 * 20000 * 4 / 1e9 - r["in"]) < 1.0
    assert abs(450 * 2000 * 20000 * 4 / 1e9 - r["out"]) < 0.01


def test_oracle_digests_are_frozen():
    """Regression guard: tests/golden/oracle_digests.json (written by
    tests/golden/make_oracle_golden.py from oracle/ only)."""
    import hashlib
    with open(os.path.join(GOLDEN, "oracle_digests.json")) as f:
        dig = json.load(f)
    for s in TABLE_SETUPS:
        t = table(s)
        assert hashlib.sha256(np.ascontiguousarray(t).tobytes()).hexdigest() == dig["tables"][s.name]["sha256"]
    s = wl.TINY
    t = table(s)
    g = dig["tiny_output"]
    x = wl.make_input(s, s.nr_samples + int(t.max()), g["in_pitch"], pulse_shifts=t[64])
    o = oracle.dedisperse(x, t, s.nr_samples)[0]
    assert hashlib.sha256(o.astype(np.float32).tobytes()).hexdigest() == g["sha256_f32"]
    assert list(np.unravel_index(np.argmax(o), o.shape)) == g["argmax"] == [64, 300]
