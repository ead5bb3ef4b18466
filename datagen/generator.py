"""ctypes front-end of datagen/dg.c (seeded filterbank generator)."""
from __future__ import annotations

import ctypes
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "dg.c"
_LIB = _HERE / "libdg.so"
_lib = None


class _Pulse(ctypes.Structure):
    _fields_ = [("t0", ctypes.c_int64), ("width", ctypes.c_int64), ("amp", ctypes.c_double)]


def lib_path() -> Path:
    return _LIB


def build(force: bool = False) -> Path:
    """Compile dg.c into datagen/libdg.so (gcc -O2 -fopenmp); no-op when up to date."""
    if force or not _LIB.exists() or _LIB.stat().st_mtime < _SRC.stat().st_mtime:
        tmp = _LIB.with_suffix(f".so.tmp{os.getpid()}")
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-o", str(tmp), str(_SRC), "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        build()
        lib = ctypes.CDLL(str(_LIB))
        lib.dg_fill.restype = None
        lib.dg_fill.argtypes = [ctypes.c_void_p, ctypes.c_size_t, ctypes.c_int32, ctypes.c_int64, ctypes.c_int64,
                                ctypes.c_uint64, ctypes.c_double, ctypes.c_double, ctypes.c_int32,
                                ctypes.c_void_p, ctypes.c_void_p]
        lib.dg_fill16.restype = None
        lib.dg_fill16.argtypes = [ctypes.c_void_p, ctypes.c_size_t, ctypes.c_int32, ctypes.c_int64, ctypes.c_int64,
                                  ctypes.c_uint64, ctypes.c_double, ctypes.c_double, ctypes.c_double, ctypes.c_int32,
                                  ctypes.c_void_p, ctypes.c_void_p]
        lib.dg_checksum.restype = ctypes.c_uint64
        lib.dg_checksum.argtypes = [ctypes.c_void_p, ctypes.c_size_t, ctypes.c_int32, ctypes.c_int64]
        _lib = lib
    return _lib


def generate(seed: int, nchans: int, nsamp: int, pulses=(), pulse_delays=None, *, t_begin: int = 0,
             mean: float = 127.0, sigma: float = 16.0, out: np.ndarray | None = None, bits: int = 8,
             max_value: int | None = None) -> np.ndarray:
    """Return x[nchans][nsamp] for absolute samples [t_begin, t_begin+nsamp): uint8 (bits = 8), or uint16 clipped to
    [0, max_value] (bits = 16; max_value = the stated bit depth, default 65535).

    ``pulses`` is a sequence of (t0, width, amp); ``pulse_delays`` an int64 array [npulses][nchans] of the
    per-channel arrival offsets in samples (computed by the caller, e.g. ``workloads.pulse_sweep``).
    ``out`` may be any C-contiguous-rows uint8 array (e.g. a view of pinned memory) with shape
    [nchans][>=nsamp]; its row stride is honoured.
    """
    lib = _load()
    dt = np.uint16 if bits == 16 else np.uint8
    assert bits in (8, 16)
    if out is None:
        out = np.empty((nchans, nsamp), dtype=dt)
    assert out.dtype == dt and out.shape[0] == nchans and out.shape[1] >= nsamp and out.strides[1] == out.itemsize
    npulses = len(pulses)
    if npulses:
        parr = (_Pulse * npulses)(*[_Pulse(int(p[0]), int(p[1]), float(p[2])) for p in pulses])
        pd = np.ascontiguousarray(pulse_delays, dtype=np.int64)
        assert pd.shape == (npulses, nchans)
        pptr, dptr = ctypes.addressof(parr), pd.ctypes.data
    else:
        pptr, dptr = None, None
    if bits == 16:
        lib.dg_fill16(out.ctypes.data, out.strides[0], nchans, t_begin, nsamp, seed, mean, sigma,
                      float(65535 if max_value is None else max_value), npulses, pptr, dptr)
    else:
        lib.dg_fill(out.ctypes.data, out.strides[0], nchans, t_begin, nsamp, seed, mean, sigma, npulses, pptr, dptr)
    return out


def checksum(x: np.ndarray) -> int:
    assert x.dtype in (np.uint8, np.uint16) and x.ndim == 2 and x.strides[1] == x.itemsize
    return int(_load().dg_checksum(x.ctypes.data, x.strides[0], x.shape[0], x.shape[1] * x.itemsize))
