"""ctypes loader of the ORACLE (oracle/oracle.cpp) — test infrastructure only.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` / ``--impl reference`` legs may
import this package. The product package never does, and this package never imports the product.
Every function here is a thin wrapper; the arithmetic is in oracle.cpp (cited there).
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "oracle.cpp"
_LIB = _HERE / "liboracle.so"
_lib = None

CAND_DTYPE = np.dtype([("sample", np.uint64), ("dm", np.float32), ("snr", np.float32),
                       ("width", np.uint32), ("range", np.uint32), ("dm_index", np.uint32)], align=True)


def build(force: bool = False) -> Path:
    """g++ -O2 -ffp-contract=off, single-threaded; no-op when up to date."""
    if force or not _LIB.exists() or _LIB.stat().st_mtime < _SRC.stat().st_mtime:
        tmp = _LIB.with_suffix(f".so.tmp{os.getpid()}")
        subprocess.check_call(["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-fPIC", "-shared",
                               "-o", str(tmp), str(_SRC)])
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is not None:
        return _lib
    build()
    L = ctypes.CDLL(str(_LIB))
    vp, i32, i64, f64, sz, u64 = (ctypes.c_void_p, ctypes.c_int32, ctypes.c_int64, ctypes.c_double,
                                  ctypes.c_size_t, ctypes.c_uint64)
    L.orc_delay_constants.argtypes = [i32, vp, f64, vp]; L.orc_delay_constants.restype = None
    L.orc_dm.argtypes = [f64, f64, i32]; L.orc_dm.restype = f64
    L.orc_delay.argtypes = [f64, f64, i32]; L.orc_delay.restype = i64
    L.orc_delay_table.argtypes = [vp, i32, f64, f64, i32, i32, i32, vp]; L.orc_delay_table.restype = None
    L.orc_bin.argtypes = [vp, sz, i32, i64, i64, i32, vp]; L.orc_bin.restype = None
    L.orc_bin16.argtypes = [vp, sz, i32, i64, i64, i32, vp]; L.orc_bin16.restype = None
    L.orc_dedisperse.argtypes = [vp, i64, i32, vp, f64, f64, i32, i32, i32, i64, vp]; L.orc_dedisperse.restype = None
    L.orc_row_stats.argtypes = [vp, i64, vp, vp, vp]; L.orc_row_stats.restype = i32
    for f in (L.orc_boxcar_snr, L.orc_boxcar_snr_prefix):
        f.argtypes = [vp, i64, vp, i32, f64, f64, vp, vp]; f.restype = None
    L.orc_find_peaks.argtypes = [vp, i32, i64, f64, i32, i32, vp, vp, i64]; L.orc_find_peaks.restype = i64
    L.orc_search_rows.argtypes = [vp, i64, i32, vp, f64, f64, i32, i32, i32, i64, i64, vp, i32, f64, u64, i32, i32, i32,
                                  vp, vp, vp, vp, vp, i64]
    L.orc_boxcar_snr_perwidth.argtypes = [vp, i64, i64, vp, i32, vp, vp, vp]; L.orc_boxcar_snr_perwidth.restype = None
    L.orc_search_rows.restype = i64
    L.orc_range_max_delay_unbinned.argtypes = [vp, i32, f64, f64, i32, i32]; L.orc_range_max_delay_unbinned.restype = i64
    _lib = L
    return L


def _p(a):
    return None if a is None else a.ctypes.data


def delay_constants(freq_mhz, tsamp_s) -> np.ndarray:
    f = np.ascontiguousarray(freq_mhz, dtype=np.float64)
    k = np.empty_like(f)
    _load().orc_delay_constants(len(f), _p(f), float(tsamp_s), _p(k))
    return k


def dm_value(dm_low, dm_step, i) -> float:
    return float(_load().orc_dm(float(dm_low), float(dm_step), int(i)))


def delay(k_c, dm, bin_=1) -> int:
    return int(_load().orc_delay(float(k_c), float(dm), int(bin_)))


def delay_table(k: np.ndarray, rng, i0: int = 0, i1: int | None = None) -> np.ndarray:
    """delay(c, i) in binned samples for rows [i0, i1) of rng = (dm_low, dm_step, ndms, bin): int64 [i1-i0][nchans]."""
    k = np.ascontiguousarray(k, dtype=np.float64)
    i1 = rng[2] if i1 is None else i1
    out = np.empty((i1 - i0, len(k)), dtype=np.int64)
    _load().orc_delay_table(_p(k), len(k), float(rng[0]), float(rng[1]), int(rng[3]), i0, i1, _p(out))
    return out


def bin_time(x: np.ndarray, start: int, nbinned: int, b: int, out: np.ndarray | None = None) -> np.ndarray:
    """x: uint8 or uint16 samples [nchans][nsamp] (16-bit input: b * max(x) must fit uint16, checked here)."""
    assert x.dtype in (np.uint8, np.uint16) and x.ndim == 2 and x.strides[1] == x.itemsize
    assert start + nbinned * b <= x.shape[1]
    if out is None:
        out = np.empty((x.shape[0], nbinned), dtype=np.uint16)
    assert out.dtype == np.uint16 and out.shape == (x.shape[0], nbinned) and out.flags.c_contiguous
    if x.dtype == np.uint16:
        if x.size:
            assert int(x[:, start:start + nbinned * b].max()) * b <= 65535, "binned 16-bit samples must fit uint16"
        _load().orc_bin16(_p(x), x.strides[0], x.shape[0], start, nbinned, b, _p(out))
    else:
        _load().orc_bin(_p(x), x.strides[0], x.shape[0], start, nbinned, b, _p(out))
    return out


def dedisperse(xb: np.ndarray, k: np.ndarray, rng, i0: int, i1: int, T: int) -> np.ndarray:
    """rng = (dm_low, dm_step, ndms, bin). Returns D[(i1-i0)][T] int64."""
    assert xb.dtype == np.uint16 and xb.flags.c_contiguous
    D = np.empty((i1 - i0, T), dtype=np.int64)
    _load().orc_dedisperse(_p(xb), xb.shape[1], xb.shape[0], _p(k), rng[0], rng[1], rng[3], i0, i1, T, _p(D))
    return D


def row_stats(row: np.ndarray):
    """Returns (mu, sigma, n, iterations, lo, hi, degenerate)."""
    row = np.ascontiguousarray(row, dtype=np.int64)
    mu, sg = ctypes.c_double(), ctypes.c_double()
    info = np.zeros(4, dtype=np.int64)
    rc = _load().orc_row_stats(_p(row), len(row), ctypes.addressof(mu), ctypes.addressof(sg), _p(info))
    return mu.value, sg.value, int(info[0]), int(info[1]), int(info[2]), int(info[3]), bool(rc)


def boxcar_snr(row: np.ndarray, widths, mu: float, sigma: float, prefix: bool = False):
    row = np.ascontiguousarray(row, dtype=np.int64)
    w = np.ascontiguousarray(widths, dtype=np.int32)
    S = np.empty(len(row), dtype=np.float64)
    wb = np.empty(len(row), dtype=np.int32)
    fn = _load().orc_boxcar_snr_prefix if prefix else _load().orc_boxcar_snr
    fn(_p(row), len(row), _p(w), len(w), float(mu), float(sigma), _p(S), _p(wb))
    return S, wb


def boxcar_snr_perwidth(row: np.ndarray, T: int, widths):
    """Reading C7m: per-width measured statistics. row holds Tx >= T samples (Tx - T = E of reading C3x). Returns
    (S[T], wbest[T], wstats[nwidths][3] = mu_w, sigma_w, p_w)."""
    row = np.ascontiguousarray(row, dtype=np.int64)
    w = np.ascontiguousarray(widths, dtype=np.int32)
    S = np.empty(T, dtype=np.float64)
    wb = np.empty(T, dtype=np.int32)
    ws = np.zeros((len(w), 3), dtype=np.float64)
    _load().orc_boxcar_snr_perwidth(_p(row), int(T), len(row), _p(w), len(w), _p(S), _p(wb), _p(ws))
    return S, wb, ws


def find_peaks(S: np.ndarray, threshold: float, r0: int = 0, r1: int | None = None, cap: int = 1 << 20):
    S = np.ascontiguousarray(S, dtype=np.float64)
    nrows, T = S.shape
    r1 = nrows if r1 is None else r1
    rr = np.empty(cap, dtype=np.int32); tt = np.empty(cap, dtype=np.int64)
    n = int(_load().orc_find_peaks(_p(S), nrows, T, float(threshold), r0, r1, _p(rr), _p(tt), cap))
    assert n <= cap, "raise cap"
    return rr[:n].copy(), tt[:n].copy()


def range_max_delay_unbinned(k, rng) -> int:
    return int(_load().orc_range_max_delay_unbinned(_p(k), len(k), rng[0], rng[1], rng[2], rng[3]))


def chunk_geometry(k: np.ndarray, ranges, nsamp_total: int, chunk_len: int | None = None, boxcar_extra: int = 0):
    """Reading C3: overlap S = max_r S_r rounded up to a multiple of B = max bin; chunk input
    length L (multiple of B, > S), n_out = L - S, chunk j starts at j*n_out; the last chunk takes the remaining
    input rounded down to a multiple of B. Returns dict(B, S, L, n_out, chunks=[(start, L_j, n_out_j)]).
    boxcar_extra = E > 0 is reading C3x (boxcar-complete chunks): every row is dedispersed E binned samples beyond its
    chunk's output span, so S_r = b_r * (delay(C-1, r, last) + E)."""
    B = max(r[3] for r in ranges)
    S = max(range_max_delay_unbinned(k, r) + r[3] * boxcar_extra for r in ranges)
    S = -(-S // B) * B
    L = (nsamp_total // B) * B if chunk_len is None else chunk_len
    assert L % B == 0 and L > S
    n_out = L - S
    chunks, start = [], 0
    while True:
        rem = ((nsamp_total - start) // B) * B
        if rem <= S:
            break
        Lj = min(L, rem)
        chunks.append((start, Lj, Lj - S))
        if Lj < L or start + Lj >= (nsamp_total // B) * B:
            break
        start += n_out
    return dict(B=B, S=S, L=L, n_out=n_out, chunks=chunks)


def search_rows(xb: np.ndarray, k: np.ndarray, rng, range_index: int, T: int, widths, threshold: float,
                chunk_start: int, i0: int, i1: int, want=("D", "stats"), cap: int = 1 << 20, extra: int = 0,
                per_width: bool = False):
    """Steps a4..a7 for rows [i0,i1) of one range on one binned chunk. Returns dict with 'cands' (structured array,
    canonical order) and whichever of 'D','stats','S','w' were asked for. extra = E (reading C3x): rows are dedispersed for
    T + E samples ('D' then has T + E columns), statistics / S / peaks stay on the first T. per_width: reading C7m
    (each width normalised by the measured statistics of its own boxcar series) instead of C7."""
    assert xb.dtype == np.uint16 and xb.flags.c_contiguous
    w = np.ascontiguousarray(widths, dtype=np.int32)
    n = i1 - i0
    D = np.empty((n, T + extra), np.int64) if "D" in want else None
    st = np.empty((n, 2), np.float64) if "stats" in want else None
    S = np.empty((n, T), np.float64) if "S" in want else None
    W = np.empty((n, T), np.int32) if "w" in want else None
    c = np.zeros(cap, dtype=CAND_DTYPE)
    cnt = int(_load().orc_search_rows(_p(xb), xb.shape[1], xb.shape[0], _p(k), rng[0], rng[1], rng[2], rng[3],
                                      range_index, T, int(extra), _p(w), len(w), float(threshold), int(chunk_start), i0, i1,
                                      1 if per_width else 0, _p(D), _p(st), _p(S), _p(W), _p(c), cap))
    assert cnt <= cap, "raise cap"
    out = dict(cands=c[:cnt].copy(), count=cnt)
    if D is not None: out["D"] = D
    if st is not None: out["stats"] = st
    if S is not None: out["S"] = S
    if W is not None: out["w"] = W
    return out


def cluster_candidates(cands: np.ndarray, dm_tol: float, gap: int):
    """Reading C10, the definition written out in O(n^2): candidates a, b are linked iff |dm_a - dm_b| <= dm_tol
    and sample_a <= sample_b + width_b + gap and sample_b <= sample_a + width_a + gap; clusters are the connected
    components. Returns a list of clusters, each a sorted list of member indices, plus the representative index of each
    (highest snr; first by (range, dm_index, sample) on ties). Pure Python: small lists only."""
    n = len(cands)
    s = [int(v) for v in cands["sample"]]
    w = [int(v) for v in cands["width"]]
    dm = [float(v) for v in cands["dm"]]
    adj = [[] for _ in range(n)]
    for a in range(n):
        for b in range(a + 1, n):
            if abs(dm[a] - dm[b]) <= dm_tol and s[a] <= s[b] + w[b] + gap and s[b] <= s[a] + w[a] + gap:
                adj[a].append(b)
                adj[b].append(a)
    seen, clusters = [False] * n, []
    for a in range(n):
        if seen[a]:
            continue
        comp, stack = [], [a]
        seen[a] = True
        while stack:
            u = stack.pop()
            comp.append(u)
            for v in adj[u]:
                if not seen[v]:
                    seen[v] = True
                    stack.append(v)
        clusters.append(sorted(comp))
    key = lambda i: (-float(cands["snr"][i]), int(cands["range"][i]), int(cands["dm_index"][i]), int(cands["sample"][i]))
    reps = [min(c, key=key) for c in clusters]
    return clusters, reps
