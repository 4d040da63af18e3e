"""CPU oracle for brute-force dedispersion -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Thin ctypes wrapper over ``oracle/dedisp_oracle.c`` (Algorithm 1 and Eq. (1) of
arXiv 1601.01165).  Only ``tests/``, ``__graft_entry__.smoke()``
and ``bench.py``'s ``cpu_baseline`` / ``--impl reference`` legs may import this
package.  It imports nothing from ``paper_1601_01165_b200`` and shares no code
with the CUDA path.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
import threading

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "dedisp_oracle.c")
_LIB = os.path.join(_HERE, "libdedisp_oracle.so")
_lock = threading.Lock()
_lib = None

CFLAGS = ["-O2", "-fopenmp", "-ffp-contract=off", "-fno-fast-math", "-shared", "-fPIC"]


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (building the checker is not using it)."""
    if (not force and os.path.exists(_LIB)
            and os.path.getmtime(_LIB) >= os.path.getmtime(_SRC)):
        return _LIB
    tmp = _LIB + ".tmp.%d" % os.getpid()
    subprocess.run(["gcc", *CFLAGS, "-o", tmp, _SRC, "-lm"], check=True)
    os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    with _lock:
        if _lib is not None:
            return _lib
        lib = ctypes.CDLL(build())
        c_int, c_i64, c_dbl, vp = ctypes.c_int, ctypes.c_int64, ctypes.c_double, ctypes.c_void_p
        lib.oracle_channel_freq_MHz.restype = c_dbl
        lib.oracle_channel_freq_MHz.argtypes = [c_dbl, c_dbl, c_int]
        lib.oracle_f_high_MHz.restype = c_dbl
        lib.oracle_f_high_MHz.argtypes = [c_dbl, c_dbl, c_int]
        lib.oracle_trial_dm.restype = c_dbl
        lib.oracle_trial_dm.argtypes = [c_dbl, c_dbl, c_int]
        lib.oracle_delay_samples.restype = c_dbl
        lib.oracle_delay_samples.argtypes = [c_dbl, c_dbl, c_dbl, c_dbl]
        lib.oracle_round_half_up.restype = c_i64
        lib.oracle_round_half_up.argtypes = [c_dbl]
        lib.oracle_shift_table.restype = c_int
        lib.oracle_shift_table.argtypes = [c_int, c_dbl, c_dbl, c_dbl, c_dbl, c_dbl, c_int, vp]
        lib.oracle_dedisperse_f32.restype = None
        lib.oracle_dedisperse_f32.argtypes = [vp, c_i64, c_int, c_int, c_i64, vp, c_int, vp, vp]
        lib.oracle_dedisperse_u8.restype = None
        lib.oracle_dedisperse_u8.argtypes = [vp, c_i64, c_int, c_int, c_i64, vp, c_int, vp]
        lib.oracle_dedisperse_f32_points.restype = None
        lib.oracle_dedisperse_f32_points.argtypes = [vp, c_i64, c_int, vp, vp, c_i64, vp, vp]
        lib.oracle_dedisperse_u8_points.restype = None
        lib.oracle_dedisperse_u8_points.argtypes = [vp, c_i64, c_int, vp, vp, c_i64, vp]
        lib.oracle_num_threads.restype = c_int
        lib.oracle_set_num_threads.argtypes = [c_int]
        _lib = lib
        return lib


def _ptr(a: np.ndarray):
    return a.ctypes.data_as(ctypes.c_void_p)


# ---- Eq. (1) ---------------------------------------------------------------

def channel_freq_MHz(f_low_MHz, channel_bw_MHz, c):
    return _load().oracle_channel_freq_MHz(f_low_MHz, channel_bw_MHz, int(c))


def f_high_MHz(f_low_MHz, channel_bw_MHz, nr_channels):
    return _load().oracle_f_high_MHz(f_low_MHz, channel_bw_MHz, int(nr_channels))


def trial_dm(dm_first, dm_step, i):
    return _load().oracle_trial_dm(dm_first, dm_step, int(i))


def delay_samples(f_MHz, f_h_MHz, dm, sample_rate):
    """Eq. (1) times the sample rate, before rounding."""
    return _load().oracle_delay_samples(f_MHz, f_h_MHz, dm, sample_rate)


def round_half_up(x):
    return _load().oracle_round_half_up(x)


def shift_of(f_MHz, f_h_MHz, dm, sample_rate):
    """shift as a function of frequency: used for the 'zero at f_h' pin."""
    return round_half_up(delay_samples(f_MHz, f_h_MHz, dm, sample_rate))


def shift_table(nr_channels, f_low_MHz, channel_bw_MHz, sample_rate, dm_first, dm_step,
                nr_dms) -> np.ndarray:
    """int32 [nr_dms][nr_channels] table of Delta(chan, dm)."""
    out = np.empty((nr_dms, nr_channels), dtype=np.int32)
    rc = _load().oracle_shift_table(int(nr_channels), f_low_MHz, channel_bw_MHz, sample_rate,
                                    dm_first, dm_step, int(nr_dms), _ptr(out))
    if rc != 0:
        raise OverflowError("shift does not fit int32")
    return out


# ---- Algorithm 1 -----------------------------------------------------------

def _check_in(x, shift, nr_samples):
    if x.ndim == 2:
        x = x[None]
    assert x.ndim == 3 and x.flags.c_contiguous
    shift = np.ascontiguousarray(shift, dtype=np.int32)
    nr_dms, nr_channels = shift.shape
    assert x.shape[1] == nr_channels, "input rows are channels (PAPER.md:45)"
    assert shift.min() >= 0 and nr_samples + int(shift.max()) <= x.shape[2], \
        "reads must stay inside the padded row"
    return x, shift, nr_dms, nr_channels


def dedisperse(x: np.ndarray, shift: np.ndarray, nr_samples: int, want_sabs: bool = False):
    """out[b][dm][t] = sum_c x[b][c][t + shift[dm][c]]  (Algorithm 1).

    x: float32 or uint8, [B][C][pitch] (or [C][pitch]).  Returns float64 (f32
    input) or uint64 (u8 input) of shape [B][D][S]; with want_sabs also the
    float64 sum of |x| per output (for the fp32 tolerance).
    """
    x, shift, nr_dms, nr_channels = _check_in(x, shift, nr_samples)
    B, _, pitch = x.shape
    lib = _load()
    if x.dtype == np.float32:
        out = np.empty((B, nr_dms, nr_samples), dtype=np.float64)
        sabs = np.empty_like(out) if want_sabs else None
        lib.oracle_dedisperse_f32(_ptr(x), pitch, nr_channels, nr_dms, nr_samples, _ptr(shift), B,
                                  _ptr(out), _ptr(sabs) if want_sabs else None)
        return (out, sabs) if want_sabs else out
    if x.dtype == np.uint8:
        out = np.empty((B, nr_dms, nr_samples), dtype=np.uint64)
        lib.oracle_dedisperse_u8(_ptr(x), pitch, nr_channels, nr_dms, nr_samples, _ptr(shift), B,
                                 _ptr(out))
        return (out, None) if want_sabs else out
    raise TypeError("input must be float32 or uint8")


def dedisperse_points(x: np.ndarray, shift: np.ndarray, nr_samples: int, pts: np.ndarray,
                      want_sabs: bool = False):
    """The same sums at pts = [[beam, dm, sample], ...] only."""
    x, shift, nr_dms, nr_channels = _check_in(x, shift, nr_samples)
    B, _, pitch = x.shape
    pts = np.ascontiguousarray(pts, dtype=np.int64).reshape(-1, 3)
    assert (pts >= 0).all() and (pts[:, 0] < B).all() and (pts[:, 1] < nr_dms).all() \
        and (pts[:, 2] < nr_samples).all()
    n = pts.shape[0]
    lib = _load()
    if x.dtype == np.float32:
        out = np.empty(n, dtype=np.float64)
        sabs = np.empty(n, dtype=np.float64) if want_sabs else None
        lib.oracle_dedisperse_f32_points(_ptr(x), pitch, nr_channels, _ptr(shift), _ptr(pts), n,
                                         _ptr(out), _ptr(sabs) if want_sabs else None)
        return (out, sabs) if want_sabs else out
    if x.dtype == np.uint8:
        out = np.empty(n, dtype=np.uint64)
        lib.oracle_dedisperse_u8_points(_ptr(x), pitch, nr_channels, _ptr(shift), _ptr(pts), n,
                                        _ptr(out))
        return (out, None) if want_sabs else out
    raise TypeError("input must be float32 or uint8")


def num_threads() -> int:
    return _load().oracle_num_threads()


def set_num_threads(n: int) -> None:
    _load().oracle_set_num_threads(int(n))
