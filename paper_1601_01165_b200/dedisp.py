"""Thin ctypes binding over libdedisp_b200.so (include/dedisp.h): argument marshalling only.

Every step of the path runs in the library's CUDA kernels.  There is no CPU fallback: if the
library is missing or there is no device the calls raise.  PyTorch is used by callers for device
memory and streams; this module accepts torch tensors, NumPy arrays (host entry point) or raw
integer addresses.
"""
from __future__ import annotations

import ctypes
import os
from typing import Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libdedisp_b200.so")

F32, U8 = 0, 1
(MAX_SHIFT, IN_SAMPLES, IN_PITCH, OUT_PITCH, VARIANT, NR_CHANNELS, NR_DMS, NR_SAMPLES, IN_DTYPE,
 MAX_STEP, RESERVED_BEAMS, PAIR_PITCH, STREAM_H2D_BYTES) = range(13)

# every symbol include/dedisp.h declares
SYMBOLS = [
    "dedisp_plan_create", "dedisp_plan_reserve", "dedisp_shift_table", "dedisp_plan_get", "dedisp_execute",
    "dedisp_execute_variant", "dedisp_execute_static_scratch", "dedisp_static_scratch_bytes", "dedisp_execute_host", "dedisp_execute_host_async", "dedisp_host_sync",
    "dedisp_stream_block_async", "dedisp_stream_reset",
    "dedisp_plan_destroy", "dedisp_variant_count",
    "dedisp_variant_name", "dedisp_variant_supported", "dedisp_plan_set_variant", "dedisp_tune",
    "dedisp_plan_load_tuning", "dedisp_status_string", "dedisp_last_error",
]

_lib = None


class DedispError(RuntimeError):
    def __init__(self, status: int, msg: str):
        super().__init__(msg)
        self.status = status


def load_library() -> ctypes.CDLL:
    """dlopen the in-tree library (build it first: python -m paper_1601_01165_b200.build)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError("%s not built: run `python -m paper_1601_01165_b200.build` "
                          "(there is no CPU fallback)" % LIB_PATH)
    lib = ctypes.CDLL(LIB_PATH)
    vp, ci, i64, dbl = ctypes.c_void_p, ctypes.c_int, ctypes.c_int64, ctypes.c_double
    lib.dedisp_plan_create.argtypes = [ctypes.POINTER(vp), ci, dbl, dbl, dbl, i64, dbl, dbl, ci, ci]
    lib.dedisp_plan_reserve.argtypes = [vp, ci]
    lib.dedisp_shift_table.argtypes = [vp, vp]
    lib.dedisp_plan_get.argtypes = [vp, ci, ctypes.POINTER(i64)]
    lib.dedisp_execute.argtypes = [vp, vp, vp, ci, vp]
    lib.dedisp_execute_variant.argtypes = [vp, ci, vp, vp, ci, vp]
    lib.dedisp_execute_host.argtypes = [vp, vp, vp, ci, vp]
    lib.dedisp_execute_static_scratch.argtypes = [vp, vp, vp, ci, vp]
    lib.dedisp_static_scratch_bytes.argtypes = []
    lib.dedisp_static_scratch_bytes.restype = i64
    lib.dedisp_execute_host_async.argtypes = [vp, vp, vp, ci]
    lib.dedisp_host_sync.argtypes = [vp]
    lib.dedisp_stream_block_async.argtypes = [vp, vp, i64, vp, i64, i64]
    lib.dedisp_stream_reset.argtypes = [vp]
    lib.dedisp_plan_destroy.argtypes = [vp]
    lib.dedisp_variant_count.argtypes = []
    lib.dedisp_variant_name.argtypes = [ci]
    lib.dedisp_variant_name.restype = ctypes.c_char_p
    lib.dedisp_variant_supported.argtypes = [vp, ci]
    lib.dedisp_plan_set_variant.argtypes = [vp, ci]
    lib.dedisp_tune.argtypes = [vp, vp, vp, ci, vp, ctypes.c_char_p, vp]
    lib.dedisp_plan_load_tuning.argtypes = [vp, ctypes.c_char_p, ci, ctypes.POINTER(ci)]
    lib.dedisp_status_string.argtypes = [ci]
    lib.dedisp_status_string.restype = ctypes.c_char_p
    lib.dedisp_last_error.argtypes = []
    lib.dedisp_last_error.restype = ctypes.c_char_p
    for name in SYMBOLS:
        if getattr(lib, name).restype not in (ctypes.c_char_p, i64):
            getattr(lib, name).restype = ci
    _lib = lib
    return lib


def _check(rc: int, what: str):
    if rc != 0:
        lib = load_library()
        raise DedispError(rc, "%s: %s (%s)" % (what, lib.dedisp_status_string(rc).decode(),
                                               lib.dedisp_last_error().decode()))


def _addr(x) -> int:
    """Raw address of a torch tensor / NumPy array / int."""
    if isinstance(x, int):
        return x
    if hasattr(x, "data_ptr"):
        return x.data_ptr()
    if isinstance(x, np.ndarray):
        return x.ctypes.data
    raise TypeError("expected a torch tensor, NumPy array or integer address")


def _stream(stream) -> Optional[int]:
    if stream is None:
        return None
    return int(getattr(stream, "cuda_stream", stream)) or None


def static_scratch_bytes() -> int:
    """dedisp_static_scratch_bytes: size of the fixed scratch array execute_static_scratch works in."""
    return int(load_library().dedisp_static_scratch_bytes())


def variant_count() -> int:
    return load_library().dedisp_variant_count()


def variant_name(v: int) -> Optional[str]:
    s = load_library().dedisp_variant_name(int(v))
    return None if s is None else s.decode()


class Plan:
    """dedisp_plan_create ... dedisp_plan_destroy (see include/dedisp.h for the contract)."""

    def __init__(self, nr_channels, f_low_MHz, channel_bw_MHz, sample_rate, nr_samples, dm_first,
                 dm_step, nr_dms, in_dtype=F32):
        self._lib = load_library()
        h = ctypes.c_void_p()
        rc = self._lib.dedisp_plan_create(ctypes.byref(h), int(nr_channels), float(f_low_MHz),
                                          float(channel_bw_MHz), float(sample_rate),
                                          int(nr_samples), float(dm_first), float(dm_step),
                                          int(nr_dms), int(in_dtype))
        self._h = h if rc == 0 else None
        _check(rc, "dedisp_plan_create")

    # -- lifetime
    def destroy(self):
        if getattr(self, "_h", None) is not None:
            self._lib.dedisp_plan_destroy(self._h)
            self._h = None

    __del__ = destroy

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.destroy()

    # -- queries
    def get(self, what: int) -> int:
        v = ctypes.c_int64()
        _check(self._lib.dedisp_plan_get(self._h, int(what), ctypes.byref(v)), "dedisp_plan_get")
        return v.value

    max_shift = property(lambda self: self.get(MAX_SHIFT))
    in_samples = property(lambda self: self.get(IN_SAMPLES))
    in_pitch = property(lambda self: self.get(IN_PITCH))
    out_pitch = property(lambda self: self.get(OUT_PITCH))
    variant = property(lambda self: self.get(VARIANT))
    nr_channels = property(lambda self: self.get(NR_CHANNELS))
    nr_dms = property(lambda self: self.get(NR_DMS))
    nr_samples = property(lambda self: self.get(NR_SAMPLES))
    in_dtype = property(lambda self: self.get(IN_DTYPE))
    max_step = property(lambda self: self.get(MAX_STEP))
    reserved_beams = property(lambda self: self.get(RESERVED_BEAMS))
    pair_pitch = property(lambda self: self.get(PAIR_PITCH))
    stream_h2d_bytes = property(lambda self: self.get(STREAM_H2D_BYTES))

    def reserve(self, nr_beams: int):
        """dedisp_plan_reserve: size the uint8 pair workspace for batches of nr_beams beams."""
        _check(self._lib.dedisp_plan_reserve(self._h, int(nr_beams)), "dedisp_plan_reserve")

    def shift_table(self) -> np.ndarray:
        """dedisp_shift_table: int32 [nr_dms][nr_channels], copied from the device table."""
        out = np.empty((self.nr_dms, self.nr_channels), dtype=np.int32)
        _check(self._lib.dedisp_shift_table(self._h, out.ctypes.data), "dedisp_shift_table")
        return out

    # -- execution
    def execute(self, d_in, d_out, nr_beams: int = 1, stream=None):
        _check(self._lib.dedisp_execute(self._h, _addr(d_in), _addr(d_out), int(nr_beams),
                                        _stream(stream)), "dedisp_execute")

    def execute_variant(self, variant: int, d_in, d_out, nr_beams: int = 1, stream=None):
        _check(self._lib.dedisp_execute_variant(self._h, int(variant), _addr(d_in), _addr(d_out),
                                                int(nr_beams), _stream(stream)),
               "dedisp_execute_variant")

    def execute_static_scratch(self, d_in, d_out, nr_beams: int = 1, stream=None):
        """dedisp_execute_static_scratch: execute() for callers that cannot allocate device memory (a
        pool allocator owns it all, a real-time loop, a thread beside a global-mode graph capture).
        uint8 plans on a tree_u8 variant only; the pair scratch is a fixed array in the library image
        instead of the plan's cudaMalloc'ed workspace, so the scratch need is capped
        (static_scratch_bytes()) and all such calls on one GPU must be ordered with respect to each
        other.  Same results as execute(), bit for bit.  See include/dedisp.h."""
        _check(self._lib.dedisp_execute_static_scratch(self._h, _addr(d_in), _addr(d_out), int(nr_beams),
                                                       _stream(stream)), "dedisp_execute_static_scratch")

    def execute_host(self, h_in, h_out, nr_beams: int = 1, stream=None):
        _check(self._lib.dedisp_execute_host(self._h, _addr(h_in), _addr(h_out), int(nr_beams),
                                             _stream(stream)), "dedisp_execute_host")

    def execute_host_async(self, h_in, h_out, nr_beams: int = 1):
        """Enqueue H2D + kernels + D2H on the plan's three-stream pipeline; see host_sync()."""
        _check(self._lib.dedisp_execute_host_async(self._h, _addr(h_in), _addr(h_out), int(nr_beams)),
               "dedisp_execute_host_async")

    def stream_block_async(self, h_series, series_pitch: int, h_out, out_pitch: int, t0: int):
        """One block of a long single-beam time series (see include/dedisp.h)."""
        _check(self._lib.dedisp_stream_block_async(self._h, _addr(h_series), int(series_pitch),
                                                   _addr(h_out), int(out_pitch), int(t0)),
               "dedisp_stream_block_async")

    def stream_reset(self):
        """dedisp_stream_reset: the next stream block uploads all of its S + M input columns again."""
        _check(self._lib.dedisp_stream_reset(self._h), "dedisp_stream_reset")

    def host_sync(self):
        _check(self._lib.dedisp_host_sync(self._h), "dedisp_host_sync")

    # -- variants and tuning
    def variant_supported(self, v: int) -> bool:
        return bool(self._lib.dedisp_variant_supported(self._h, int(v)))

    def supported_variants(self):
        return [v for v in range(variant_count()) if self.variant_supported(v)]

    def set_variant(self, v: int):
        _check(self._lib.dedisp_plan_set_variant(self._h, int(v)), "dedisp_plan_set_variant")

    def tune(self, d_in, d_out, nr_beams: int = 1, stream=None, cache_path: Optional[str] = None):
        """dedisp_tune: returns {variant index: mean ms} for the supported variants."""
        ms = np.empty(variant_count(), dtype=np.float32)
        _check(self._lib.dedisp_tune(self._h, _addr(d_in), _addr(d_out), int(nr_beams),
                                     _stream(stream),
                                     None if cache_path is None else cache_path.encode(),
                                     ms.ctypes.data), "dedisp_tune")
        return {v: float(ms[v]) for v in range(len(ms)) if ms[v] >= 0}

    def load_tuning(self, cache_path: str, nr_beams: int = 1) -> bool:
        """dedisp_plan_load_tuning: True if the cache had an entry for this setup and it was applied."""
        hit = ctypes.c_int(0)
        _check(self._lib.dedisp_plan_load_tuning(self._h, cache_path.encode(), int(nr_beams),
                                                 ctypes.byref(hit)), "dedisp_plan_load_tuning")
        return bool(hit.value)
