"""ctypes binding of include/aa.h — same names, same argument order, marshalling only.

Every ``aa_*`` function below calls the C entry point of the same name. Negative status codes raise :class:`AaError`
carrying ``aa_last_error()``; progress codes (AA_OK, AA_STATUS_CHUNK_DONE, AA_STATUS_FINISHED) are returned.
PAPER.md:67 (§4): "A Python front-end delegates computationally intensive tasks to the C++ API by calling into
AstroAccelerate as a shared object library."
"""
from __future__ import annotations

import ctypes
from ctypes import POINTER, byref, c_char_p, c_double, c_float, c_int32, c_int64, c_size_t, c_uint32, c_uint64, c_void_p
from pathlib import Path

import numpy as np

__all__ = [
    "AaError", "AA_OK", "AA_STATUS_CHUNK_DONE", "AA_STATUS_FINISHED", "AA_ERR_INVALID_ARG", "AA_ERR_NOT_READY",
    "AA_ERR_BUDGET_TOO_SMALL", "AA_ERR_CUDA", "AA_ERR_CANDIDATE_OVERFLOW", "AA_ERR_ORDER", "AA_ERR_INTERNAL", "AA_ERR_RANGE",
    "aa_plan_set_input_bits",
    "CANDIDATE_DTYPE", "lib_path", "load",
    "AA_LAYOUT_CHANNEL_MAJOR", "AA_LAYOUT_TIME_MAJOR", "aa_plan_create", "aa_plan_destroy", "aa_plan_set_input_layout", "aa_plan_set_boxcar_overlap", "aa_plan_set_per_width_stats", "aa_get_row_width_stats", "aa_strategy_plan", "aa_strategy_setup", "aa_strategy_destroy", "aa_strategy_get_info",
    "aa_strategy_get_range_info", "aa_strategy_get_chunk", "aa_strategy_get_delay", "aa_strategy_describe",
    "aa_strategy_reset", "aa_strategy_shard", "aa_run_dedispersion", "aa_run_dedispersion_device", "aa_run_sps", "aa_run_pipeline", "aa_get_candidates", "aa_get_clusters", "aa_cluster_candidates", "CLUSTER_DTYPE",
    "aa_get_dedispersed_row", "aa_get_row_stats", "aa_get_row_moments", "aa_get_dedispersed_device", "aa_synchronize",
    "aa_row_moments_static", "AA_STATIC_MOMENTS_MAX_ROWS",
    "aa_measure_int_add_peak", "aa_measure_int_add_peak3", "aa_get_last_timings", "aa_get_launch_count", "aa_last_error", "aa_version",
    "Plan", "Strategy",
]

AA_OK, AA_STATUS_CHUNK_DONE, AA_STATUS_FINISHED = 0, 1, 2
AA_ERR_INVALID_ARG, AA_ERR_NOT_READY, AA_ERR_BUDGET_TOO_SMALL, AA_ERR_CUDA = -1, -2, -3, -4
AA_ERR_CANDIDATE_OVERFLOW, AA_ERR_ORDER, AA_ERR_INTERNAL, AA_ERR_RANGE = -5, -6, -7, -8
AA_LAYOUT_CHANNEL_MAJOR, AA_LAYOUT_TIME_MAJOR = 0, 1
AA_STATIC_MOMENTS_MAX_ROWS = 16384      # rows per aa_row_moments_static call (include/aa.h)

CLUSTER_DTYPE = None  # defined below CANDIDATE_DTYPE
CANDIDATE_DTYPE = np.dtype([("sample", np.uint64), ("dm", np.float32), ("snr", np.float32), ("width", np.uint32),
                            ("range", np.uint32), ("dm_index", np.uint32)], align=True)


CLUSTER_DTYPE = np.dtype([("best", CANDIDATE_DTYPE), ("members", np.uint32), ("dm_min", np.float32), ("dm_max", np.float32),
                          ("sample_min", np.uint64), ("sample_end", np.uint64)], align=True)


class AaError(RuntimeError):
    def __init__(self, status: int, message: str):
        super().__init__(f"aa_status {status}: {message}")
        self.status = status
        self.message = message


class _DmRange(ctypes.Structure):
    _fields_ = [("dm_low", c_double), ("dm_step", c_double), ("ndms", c_int32), ("bin", c_int32)]


class _RangeInfo(ctypes.Structure):
    _fields_ = [("ndms", c_int32), ("bin", c_int32), ("nt", c_int64), ("row_pitch", c_int64), ("max_delay", c_int64),
                ("dm_tile", c_int32), ("t_tile", c_int32), ("chan_block", c_int32), ("window", c_int32),
                ("boxcar_extra", c_int32)]


class _StrategyInfo(ctypes.Structure):
    _fields_ = [("ready", c_int32), ("nchans", c_int32), ("nranges", c_int32), ("nwidths", c_int32), ("max_bin", c_int32),
                ("nsamp_total", c_int64), ("overlap", c_int64), ("chunk_len", c_int64), ("n_out", c_int64),
                ("nchunks", c_int64), ("next_chunk", c_int64), ("shard_rank", c_int32), ("shard_world", c_int32),
                ("arena_bytes_used", c_size_t),
                ("arena_bytes_total", c_size_t), ("max_candidates", c_size_t), ("owns_arena", c_int32), ("input_layout", c_int32),
                ("input_bits", c_int32), ("input_max", c_uint32)]


def _struct_dict(s):
    return {name: getattr(s, name) for name, _ in s._fields_}


_LIB_PATH = Path(__file__).resolve().parent / "libaa.so"
_lib = None


def lib_path() -> Path:
    return _LIB_PATH


def load():
    """Load libaa.so. Raises (no fallback) if it has not been built."""
    global _lib
    if _lib is not None:
        return _lib
    if not _LIB_PATH.exists():
        raise ImportError(f"{_LIB_PATH} is missing: build the CUDA library first (python -m paper_1912_07704_b200.build); "
                          "there is no CPU fallback")
    L = ctypes.CDLL(str(_LIB_PATH))
    vp = c_void_p
    sig = {
        "aa_plan_create": (c_int32, [POINTER(vp), c_int32, vp, c_double, vp, c_int32, vp, c_int32, c_float]),
        "aa_plan_destroy": (None, [vp]),
        "aa_plan_set_input_layout": (c_int32, [vp, c_int32]),
        "aa_plan_set_boxcar_overlap": (c_int32, [vp, c_int32]),
        "aa_plan_set_per_width_stats": (c_int32, [vp, c_int32]),
        "aa_plan_set_input_bits": (c_int32, [vp, c_int32, c_uint32]),
        "aa_get_row_width_stats": (c_int32, [vp, c_int32, c_int32, c_int32, POINTER(c_double), POINTER(c_double), POINTER(c_int64)]),
        "aa_strategy_setup": (c_int32, [POINTER(vp), vp, c_uint64, vp, c_size_t, c_size_t, vp, vp, c_size_t, c_uint64]),
        "aa_strategy_plan": (c_int32, [POINTER(vp), vp, c_uint64, c_size_t, c_size_t, c_uint64]),
        "aa_strategy_destroy": (None, [vp]),
        "aa_strategy_get_info": (c_int32, [vp, POINTER(_StrategyInfo)]),
        "aa_strategy_get_range_info": (c_int32, [vp, c_int32, POINTER(_RangeInfo)]),
        "aa_strategy_get_chunk": (c_int32, [vp, c_int64, POINTER(c_uint64), POINTER(c_uint64), POINTER(c_uint64)]),
        "aa_strategy_get_delay": (c_int32, [vp, c_int32, c_int32, c_int32, POINTER(c_int64)]),
        "aa_strategy_describe": (c_size_t, [vp, vp, c_size_t]),
        "aa_strategy_reset": (c_int32, [vp]),
        "aa_strategy_shard": (c_int32, [vp, c_int32, c_int32]),
        "aa_run_dedispersion": (c_int32, [vp, vp, c_size_t]),
        "aa_run_dedispersion_device": (c_int32, [vp, vp, c_size_t]),
        "aa_run_sps": (c_int32, [vp]),
        "aa_run_pipeline": (c_int32, [vp, vp, c_size_t]),
        "aa_get_candidates": (c_int32, [vp, POINTER(vp), POINTER(c_size_t)]),
        "aa_get_clusters": (c_int32, [vp, c_double, c_uint64, POINTER(vp), POINTER(c_size_t)]),
        "aa_cluster_candidates": (c_int32, [vp, c_size_t, c_double, c_uint64, vp, POINTER(c_size_t)]),
        "aa_get_dedispersed_row": (c_int32, [vp, c_int32, c_int32, POINTER(vp), POINTER(c_size_t)]),
        "aa_get_row_stats": (c_int32, [vp, c_int32, c_int32, POINTER(c_double), POINTER(c_double), POINTER(c_int64), POINTER(c_int32)]),
        "aa_get_row_moments": (c_int32, [vp, c_int32, vp, vp]),
        "aa_get_dedispersed_device": (c_int32, [vp, c_int32, POINTER(vp), POINTER(c_int64)]),
        "aa_row_moments_static": (c_int32, [vp, c_int64, c_int64, c_int32, vp, vp, vp]),
        "aa_synchronize": (c_int32, [vp]),
        "aa_measure_int_add_peak": (c_int32, [vp, c_int32, POINTER(c_double), POINTER(c_double), POINTER(c_double)]),
        "aa_measure_int_add_peak3": (c_int32, [vp, c_int32, POINTER(c_double), POINTER(c_double), POINTER(c_double), POINTER(c_double)]),
        "aa_get_last_timings": (c_int32, [vp, POINTER(c_float * 5)]),
        "aa_get_launch_count": (c_int32, [vp, POINTER(c_uint64)]),
        "aa_last_error": (c_char_p, []),
        "aa_version": (c_char_p, []),
    }
    for name, (res, args) in sig.items():
        f = getattr(L, name)
        f.restype, f.argtypes = res, args
    _lib = L
    return L


def aa_last_error() -> str:
    return load().aa_last_error().decode()


def aa_version() -> str:
    return load().aa_version().decode()


def _check(status: int, allow=()) -> int:
    if status < 0 and status not in allow:
        raise AaError(status, aa_last_error())
    return status


def _ptr(x):
    """Address of host numpy memory, a device pointer given as int, or anything with data_ptr() (a torch tensor)."""
    if x is None:
        return None
    if isinstance(x, int):
        return x
    if isinstance(x, np.ndarray):
        return x.ctypes.data
    if hasattr(x, "data_ptr"):
        return x.data_ptr()
    if hasattr(x, "cuda_stream"):          # torch.cuda.Stream
        return x.cuda_stream
    raise TypeError(f"cannot take the address of {type(x)}")


# ---------------------------------------------------------------------------------------------- plan / strategy
def aa_plan_create(chan_freq_mhz, tsamp_s, ranges, boxcar_widths, snr_threshold) -> int:
    """ranges: sequence of (dm_low, dm_step, ndms, bin). Returns the opaque plan handle."""
    f = np.ascontiguousarray(chan_freq_mhz, dtype=np.float64)
    rs = (_DmRange * max(1, len(ranges)))(*[_DmRange(float(r[0]), float(r[1]), int(r[2]), int(r[3])) for r in ranges])
    w = np.ascontiguousarray(boxcar_widths, dtype=np.int32)
    out = c_void_p()
    _check(load().aa_plan_create(byref(out), len(f), f.ctypes.data, float(tsamp_s), ctypes.addressof(rs), len(ranges),
                                 w.ctypes.data, len(w), float(snr_threshold)))
    return out.value


def aa_plan_set_input_layout(plan, layout: int) -> int:
    return _check(load().aa_plan_set_input_layout(plan, int(layout)))


def aa_plan_set_boxcar_overlap(plan, on: bool) -> int:
    return _check(load().aa_plan_set_boxcar_overlap(plan, 1 if on else 0))


def aa_plan_set_input_bits(plan, bits: int, max_value: int = 0) -> int:
    return _check(load().aa_plan_set_input_bits(plan, int(bits), int(max_value)))


def aa_plan_set_per_width_stats(plan, on: bool) -> int:
    return _check(load().aa_plan_set_per_width_stats(plan, 1 if on else 0))


def aa_plan_destroy(plan) -> None:
    load().aa_plan_destroy(plan)


def aa_strategy_setup(plan, nsamp_total, device_arena=None, arena_bytes=0, budget_bytes=0, compute_stream=None,
                      copy_stream=None, max_candidates=1 << 20, chunk_len_hint=0) -> int:
    out = c_void_p()
    _check(load().aa_strategy_setup(byref(out), plan, int(nsamp_total), _ptr(device_arena), int(arena_bytes),
                                    int(budget_bytes), _ptr(compute_stream), _ptr(copy_stream), int(max_candidates),
                                    int(chunk_len_hint)))
    return out.value


def aa_strategy_plan(plan, nsamp_total, budget_bytes=0, max_candidates=1 << 20, chunk_len_hint=0) -> int:
    """Host-only strategy (ready == 0): geometry, tiling and arena size without a GPU."""
    out = c_void_p()
    _check(load().aa_strategy_plan(byref(out), plan, int(nsamp_total), int(budget_bytes), int(max_candidates), int(chunk_len_hint)))
    return out.value


def aa_strategy_destroy(strategy) -> None:
    load().aa_strategy_destroy(strategy)


def aa_strategy_get_info(strategy) -> dict:
    info = _StrategyInfo()
    _check(load().aa_strategy_get_info(strategy, byref(info)))
    return _struct_dict(info)


def aa_strategy_get_range_info(strategy, rng: int) -> dict:
    info = _RangeInfo()
    _check(load().aa_strategy_get_range_info(strategy, rng, byref(info)))
    return _struct_dict(info)


def aa_strategy_get_chunk(strategy, chunk: int):
    a, b, c = c_uint64(), c_uint64(), c_uint64()
    _check(load().aa_strategy_get_chunk(strategy, chunk, byref(a), byref(b), byref(c)))
    return a.value, b.value, c.value


def aa_strategy_get_delay(strategy, rng: int, dm_index: int, chan: int) -> int:
    d = c_int64()
    _check(load().aa_strategy_get_delay(strategy, rng, dm_index, chan, byref(d)))
    return d.value


def aa_strategy_describe(strategy) -> str:
    n = load().aa_strategy_describe(strategy, None, 0)
    buf = ctypes.create_string_buffer(n)
    load().aa_strategy_describe(strategy, ctypes.addressof(buf), n)
    return buf.value.decode()


def aa_strategy_reset(strategy) -> int:
    return _check(load().aa_strategy_reset(strategy))


def aa_strategy_shard(strategy, rank: int, world: int) -> int:
    return _check(load().aa_strategy_shard(strategy, int(rank), int(world)))


# ---------------------------------------------------------------------------------------------- pipeline
def _host_input(strategy, host_input, row_stride_bytes):
    """Marshalling checks of a host array handed to aa_run_*: the C side reads raw bytes through the pointer, so a wrong
    dtype, a transposed view or a short array would be read without any error there. Raw addresses (int) pass unchecked."""
    if isinstance(host_input, np.ndarray):
        info = aa_strategy_get_info(strategy)
        item = 2 if info.get("input_bits", 8) > 8 else 1
        want = np.uint16 if item == 2 else np.uint8
        if host_input.dtype != want:
            raise TypeError(f"host_input must be {np.dtype(want).name} (the plan's sample type), got {host_input.dtype}")
        if host_input.ndim != 2 or (host_input.shape[1] > 1 and host_input.strides[1] != item):
            raise ValueError("host_input must be 2-D with unit stride along its rows")
        rows, cols = ((info["nsamp_total"], info["nchans"]) if info["input_layout"] == AA_LAYOUT_TIME_MAJOR
                      else (info["nchans"], info["nsamp_total"]))
        if host_input.shape[0] < rows or host_input.shape[1] < cols:
            raise ValueError(f"host_input has shape {host_input.shape}, the plan's layout needs at least ({rows}, {cols})")
        if row_stride_bytes is None:
            row_stride_bytes = host_input.strides[0]
    elif row_stride_bytes is None:
        row_stride_bytes = host_input.stride(0) * host_input.element_size()
    return _ptr(host_input), int(row_stride_bytes)


def aa_run_dedispersion(strategy, host_input, row_stride_bytes=None) -> int:
    """host_input: numpy array / pinned torch tensor [nchans][nsamp_total] of the plan's sample type (or a raw host
    address together with row_stride_bytes)."""
    ptr, stride = _host_input(strategy, host_input, row_stride_bytes)
    return _check(load().aa_run_dedispersion(strategy, ptr, stride))


def aa_run_dedispersion_device(strategy, device_chunk, row_stride_bytes=None) -> int:
    if row_stride_bytes is None:
        row_stride_bytes = device_chunk.stride(0) * device_chunk.element_size()
    return _check(load().aa_run_dedispersion_device(strategy, _ptr(device_chunk), int(row_stride_bytes)))


def aa_run_sps(strategy) -> int:
    return _check(load().aa_run_sps(strategy))


def aa_run_pipeline(strategy, host_input, row_stride_bytes=None) -> int:
    """The chunk loop inside the library (one call)."""
    ptr, stride = _host_input(strategy, host_input, row_stride_bytes)
    return _check(load().aa_run_pipeline(strategy, ptr, stride))


def aa_get_candidates(strategy, allow_overflow: bool = False) -> np.ndarray:
    """All candidates so far as a structured array (a copy; canonical order)."""
    p, n = c_void_p(), c_size_t()
    _check(load().aa_get_candidates(strategy, byref(p), byref(n)), allow=(AA_ERR_CANDIDATE_OVERFLOW,) if allow_overflow else ())
    if n.value == 0:
        return np.zeros(0, dtype=CANDIDATE_DTYPE)
    buf = (ctypes.c_char * (n.value * CANDIDATE_DTYPE.itemsize)).from_address(p.value)
    return np.frombuffer(buf, dtype=CANDIDATE_DTYPE).copy()


def aa_get_clusters(strategy, dm_tol: float, gap: int, allow_overflow: bool = False) -> np.ndarray:
    """Clusters of all candidates gathered so far (a copy), see include/aa.h."""
    p, n = c_void_p(), c_size_t()
    _check(load().aa_get_clusters(strategy, float(dm_tol), int(gap), byref(p), byref(n)),
           allow=(AA_ERR_CANDIDATE_OVERFLOW,) if allow_overflow else ())
    if n.value == 0:
        return np.zeros(0, dtype=CLUSTER_DTYPE)
    buf = (ctypes.c_char * (n.value * CLUSTER_DTYPE.itemsize)).from_address(p.value)
    return np.frombuffer(buf, dtype=CLUSTER_DTYPE).copy()


def aa_cluster_candidates(cands: np.ndarray, dm_tol: float, gap: int) -> np.ndarray:
    """The same clustering on any candidate array (host only, no strategy, no GPU)."""
    c = np.ascontiguousarray(cands, dtype=CANDIDATE_DTYPE)
    out = np.zeros(len(c), dtype=CLUSTER_DTYPE)
    n = c_size_t()
    _check(load().aa_cluster_candidates(c.ctypes.data if len(c) else None, len(c), float(dm_tol), int(gap),
                                        out.ctypes.data if len(c) else None, byref(n)))
    return out[:n.value].copy()


def aa_get_dedispersed_row(strategy, rng: int, dm_index: int) -> np.ndarray:
    p, n = c_void_p(), c_size_t()
    _check(load().aa_get_dedispersed_row(strategy, rng, dm_index, byref(p), byref(n)))
    buf = (ctypes.c_int32 * n.value).from_address(p.value)
    return np.frombuffer(buf, dtype=np.int32).copy()


def aa_get_row_stats(strategy, rng: int, dm_index: int):
    mu, sg, n, it = c_double(), c_double(), c_int64(), c_int32()
    _check(load().aa_get_row_stats(strategy, rng, dm_index, byref(mu), byref(sg), byref(n), byref(it)))
    return mu.value, sg.value, n.value, it.value


def aa_get_row_width_stats(strategy, rng: int, dm_index: int, width_index: int):
    """(mu_w, sigma_w, p_w) of one plan width in one row (reading C7m plans only)."""
    mu, sg, pv = c_double(), c_double(), c_int64()
    _check(load().aa_get_row_width_stats(strategy, rng, dm_index, width_index, byref(mu), byref(sg), byref(pv)))
    return mu.value, sg.value, pv.value


def aa_get_row_moments(strategy, rng: int, ndms: int | None = None):
    """sum_t D and sum_t t*D of every row of a range. The arrays are sized from the strategy's own range info (the C side
    writes ndms values whatever the caller believes); `ndms`, if given, is only checked against it."""
    n = aa_strategy_get_range_info(strategy, rng)["ndms"]
    if ndms is not None and int(ndms) != n:
        raise ValueError(f"range {rng} has {n} DM trials, not {ndms}")
    ndms = n
    a = np.zeros(ndms, dtype=np.int64)
    b = np.zeros(ndms, dtype=np.int64)
    _check(load().aa_get_row_moments(strategy, rng, a.ctypes.data, b.ctypes.data))
    return a, b


def aa_get_dedispersed_device(strategy, rng: int):
    p, pitch = c_void_p(), c_int64()
    _check(load().aa_get_dedispersed_device(strategy, rng, byref(p), byref(pitch)))
    return p.value, pitch.value


def aa_row_moments_static(device_D, row_pitch: int, nt: int, nrows: int, stream=None):
    """sum_t D and sum_t t*D of `nrows` int32 rows in device memory (row i at device_D + i*row_pitch elements), computed
    without any device allocation: the entry point for callers that cannot call cudaMalloc (all device memory already
    handed out, or a thread that must not stall the streaming loop with an allocation's device-wide synchronisation).
    At most AA_STATIC_MOMENTS_MAX_ROWS rows per call (AaError beyond that). `device_D` is a device pointer (int) or a
    torch tensor on the current device. Calls share one built-in scratch array per GPU: do not run two at once."""
    n = max(0, int(nrows))
    a = np.zeros(n, dtype=np.int64)
    b = np.zeros(n, dtype=np.int64)
    _check(load().aa_row_moments_static(_ptr(device_D), int(row_pitch), int(nt), int(nrows), a.ctypes.data, b.ctypes.data,
                                        _ptr(stream)))
    return a, b


def aa_synchronize(strategy) -> int:
    return _check(load().aa_synchronize(strategy))


def aa_measure_int_add_peak(stream=None, millis: int = 200):
    """Returns (IADD3-only lane-adds/s, IADD3+IMAD mixed lane-adds/s, SM MHz)."""
    a, b, c = c_double(), c_double(), c_double()
    _check(load().aa_measure_int_add_peak(_ptr(stream), int(millis), byref(a), byref(b), byref(c)))
    return a.value, b.value, c.value


def aa_measure_int_add_peak3(stream=None, millis: int = 200):
    """(IADD3-only, IADD3+IMAD mixed, IMAD-only) lane-adds per second and the SM clock in MHz."""
    a, b, c, d = c_double(), c_double(), c_double(), c_double()
    _check(load().aa_measure_int_add_peak3(_ptr(stream), int(millis), byref(a), byref(b), byref(c), byref(d)))
    return a.value, b.value, c.value, d.value


def aa_get_last_timings(strategy) -> dict:
    arr = (c_float * 5)()
    _check(load().aa_get_last_timings(strategy, byref(arr)))
    return dict(zip(("bin_ms", "dedisp_ms", "stats_ms", "peaks_ms", "h2d_ms"), [float(v) for v in arr]))


def aa_get_launch_count(strategy) -> int:
    n = c_uint64()
    _check(load().aa_get_launch_count(strategy, byref(n)))
    return n.value


# ---------------------------------------------------------------------------------------------- lifetime helpers
class Plan:
    """Owns an aa_plan handle."""

    def __init__(self, chan_freq_mhz, tsamp_s, ranges, boxcar_widths, snr_threshold, time_major: bool = False,
                 boxcar_overlap: bool = False, per_width_stats: bool = False, input_bits: int = 8, input_max: int = 0):
        self.handle = aa_plan_create(chan_freq_mhz, tsamp_s, ranges, boxcar_widths, snr_threshold)
        self.ranges = [tuple(r) for r in ranges]
        if time_major:
            aa_plan_set_input_layout(self.handle, AA_LAYOUT_TIME_MAJOR)
        if boxcar_overlap:
            aa_plan_set_boxcar_overlap(self.handle, True)
        if per_width_stats:
            aa_plan_set_per_width_stats(self.handle, True)
        if input_bits != 8:
            aa_plan_set_input_bits(self.handle, input_bits, input_max)

    def close(self):
        if getattr(self, "handle", None):
            aa_plan_destroy(self.handle)
            self.handle = None

    __del__ = close


class Strategy:
    """Owns an aa_strategy handle (and keeps the lent arena tensor alive)."""

    def __init__(self, plan: Plan, nsamp_total: int, *, arena=None, budget_bytes: int = 0, compute_stream=None,
                 copy_stream=None, max_candidates: int = 1 << 20, chunk_len_hint: int = 0):
        self._arena = arena
        nbytes = 0 if arena is None else arena.numel() * arena.element_size()
        self.handle = aa_strategy_setup(plan.handle, nsamp_total, arena, nbytes, budget_bytes, compute_stream, copy_stream,
                                        max_candidates, chunk_len_hint)
        self.ranges = plan.ranges
        self.info = aa_strategy_get_info(self.handle)

    def shard(self, rank: int, world: int) -> None:
        """Own chunks rank, rank+world, ... only (replicas over time chunks, one strategy per GPU)."""
        aa_strategy_shard(self.handle, rank, world)
        self.info = aa_strategy_get_info(self.handle)

    def run(self, host_input) -> np.ndarray:
        """The paper's pipeline loop: dedispersion then SPS per chunk of this strategy's shard until
        FINISHED; returns the candidates of those chunks."""
        info = aa_strategy_get_info(self.handle)
        if info["next_chunk"] < info["nchunks"]:
            while True:
                aa_run_dedispersion(self.handle, host_input)
                if aa_run_sps(self.handle) == AA_STATUS_FINISHED:
                    break
        return aa_get_candidates(self.handle)

    def clusters(self, dm_tol: float, gap: int) -> np.ndarray:
        """Friends-of-friends clusters of the candidates gathered so far (include/aa.h, aa_get_clusters)."""
        return aa_get_clusters(self.handle, dm_tol, gap)

    def close(self):
        if getattr(self, "handle", None):
            aa_strategy_destroy(self.handle)
            self.handle = None

    __del__ = close
