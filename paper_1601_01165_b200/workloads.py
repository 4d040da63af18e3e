"""Observational setups and seeded synthetic inputs (BASELINE.json `configs`).

This module serves BOTH the CUDA path and the oracle's tests, so it holds none
of the method's arithmetic: no delay formula, no shifted sum.  Anything that
depends on the shift table (row length S+M, where the test pulse goes) is passed
in by the caller.  Recipe: SURVEY.md section 8(d) / DESIGN.md "Input recipe";
shapes follow the paper's Table 2 setups.
"""
from __future__ import annotations

from dataclasses import dataclass, replace
from typing import Optional

import numpy as np

F32 = 0  # fp32 in -> fp32 out   ("All data are single precision")
U8 = 1   # uint8 in -> uint32 out (BASELINE.json config 4; not in the paper)


@dataclass(frozen=True)
class Setup:
    name: str
    nr_channels: int
    f_low_MHz: float
    channel_bw_MHz: float
    sample_rate: float
    nr_samples: int          # output samples per beam, S
    dm_first: float
    dm_step: float
    nr_dms: int
    in_dtype: int = F32
    nr_beams: int = 1
    seed: int = 0
    values: str = "gauss"    # "gauss" | "int16" (integers 0..15 as fp32) | "u8"
    pulse: Optional[tuple] = None   # (dm_index, arrival sample, amplitude)

    @property
    def seconds_of_data(self) -> float:
        return self.nr_samples / self.sample_rate

    @property
    def adds_per_beam(self) -> int:
        """One add per (dm, sample, channel): the paper's flop count
        ("20 MFLOP per DM" = 20000 x 1024 for Apertif)."""
        return self.nr_dms * self.nr_channels * self.nr_samples

    @property
    def np_in_dtype(self):
        return np.uint8 if self.in_dtype == U8 else np.float32

    @property
    def np_out_dtype(self):
        return np.uint32 if self.in_dtype == U8 else np.float32

    def plan_args(self):
        return (self.nr_channels, self.f_low_MHz, self.channel_bw_MHz, self.sample_rate,
                self.nr_samples, self.dm_first, self.dm_step, self.nr_dms, self.in_dtype)

    def table_args(self):
        return (self.nr_channels, self.f_low_MHz, self.channel_bw_MHz, self.sample_rate,
                self.dm_first, self.dm_step, self.nr_dms)


# The five BASELINE.json configs, in order.
TINY = Setup("tiny", 32, 1420.0, 1.0, 1000.0, 1024, 0.0, 1.0, 128,
             seed=160101165, values="int16", pulse=(64, 300, 100.0))
APERTIF = Setup("apertif", 1024, 1420.0, 300.0 / 1024, 20000.0, 20000, 0.0, 0.25, 2048,
                seed=160101166)
LOFAR = Setup("lofar", 32, 138.0, 6.0 / 32, 200000.0, 200000, 0.0, 0.01, 2048,
              seed=160101167)
SURVEY8 = Setup("survey8", 1536, 1220.0, 300.0 / 1536, 24414.0, 49152, 0.0, 0.2, 4096,
                in_dtype=U8, seed=160101168, values="u8")
BATCH40 = replace(APERTIF, name="batch40", nr_beams=40, seed=160101170)

CONFIGS = {s.name: s for s in (TINY, APERTIF, LOFAR, SURVEY8, BATCH40)}

# The paper's own two setups at their largest instance (Table 2 and the 12 input
# instances of 2-4096 DMs: "DMs from 0, step 0.25" for both).  Apertif: 20 kHz sampling, 300 MHz in 1024
# channels above 1420 MHz, 4096 DMs.  LOFAR: 200 kHz sampling, 6 MHz in 32 channels above 138 MHz; 2048 DMs
# is the largest instance whose input row (S + M = 0.2 M + 1.82 M samples) is still a few hundred MB.
# SURVEY.md 8(f) row 2; not BASELINE.json configs, so they are kept apart from CONFIGS.
APERTIF_PAPER = Setup("apertif_paper", 1024, 1420.0, 300.0 / 1024, 20000.0, 20000, 0.0, 0.25, 4096,
                      seed=160101171)
LOFAR_PAPER = Setup("lofar_paper", 32, 138.0, 6.0 / 32, 200000.0, 200000, 0.0, 0.25, 2048,
                    seed=160101172)
PAPER_SETUPS = {s.name: s for s in (APERTIF_PAPER, LOFAR_PAPER)}
ALL = {**CONFIGS, **PAPER_SETUPS}


def scaled(setup: Setup, **kw) -> Setup:
    """A smaller/larger variant of a setup (same band and DM grid unless overridden)."""
    return replace(setup, **kw)


def make_input(setup: Setup, in_samples: int, in_pitch: int,
               pulse_shifts: Optional[np.ndarray] = None,
               beams: Optional[range] = None) -> np.ndarray:
    """Seeded input [B][C][in_pitch]; samples [0, in_samples) of every row are
    drawn from the RNG (nothing is zero-filled: reading A8).  The pitch padding is
    POISONED (NaN for fp32, 255 for uint8): the contract says it is ignored, so a
    kernel that lets it reach an output shows up in every parity test.

    Beam b of a multi-beam setup uses seed + b, so any subset of beams can be
    regenerated.  pulse_shifts: int array [C], the shifts of setup.pulse's DM row,
    supplied by whoever owns a shift table (reading A13).
    """
    assert in_pitch >= in_samples
    beams = range(setup.nr_beams) if beams is None else beams
    C = setup.nr_channels
    x = np.full((len(beams), C, in_pitch), 255 if setup.in_dtype == U8 else np.nan,
                dtype=setup.np_in_dtype)
    for k, b in enumerate(beams):
        rng = np.random.default_rng(setup.seed + b)
        if setup.values == "gauss":
            x[k, :, :in_samples] = rng.standard_normal((C, in_samples), dtype=np.float32)
        elif setup.values == "int16":
            x[k, :, :in_samples] = rng.integers(0, 16, size=(C, in_samples)).astype(np.float32)
        elif setup.values == "u8":
            x[k, :, :in_samples] = rng.integers(0, 256, size=(C, in_samples), dtype=np.uint8)
        else:
            raise ValueError(setup.values)
        if setup.pulse is not None:
            assert pulse_shifts is not None, "pulse placement needs the DM row's shifts"
            _, t_arrival, amp = setup.pulse
            idx = t_arrival + np.asarray(pulse_shifts, dtype=np.int64)
            x[k, np.arange(C), idx] += np.asarray(amp, dtype=x.dtype)
    return x


def sample_points(setup: Setup, n: int, seed: int = 12345) -> np.ndarray:
    """n random (beam, dm, sample) output coordinates plus the corners, int64 [m][3]."""
    rng = np.random.default_rng(seed)
    B, D, S = setup.nr_beams, setup.nr_dms, setup.nr_samples
    pts = np.stack([rng.integers(0, B, n), rng.integers(0, D, n), rng.integers(0, S, n)], axis=1)
    corners = [(b, d, s) for b in {0, B - 1} for d in {0, D - 1} for s in {0, S - 1}]
    return np.concatenate([np.asarray(corners, dtype=np.int64), pts.astype(np.int64)], axis=0)
