"""Shared helpers of the GPU parity tests: run the CUDA path through the C-ABI binding and the oracle on the same
seeded bytes, and compare element by element. Only tests may import both sides."""
from __future__ import annotations

import numpy as np

import datagen
import oracle


def make_input(w, pinned: bool = False):
    pl, dms, dl = w.pulses()
    if pinned:
        import torch
        t = torch.empty((w.nchans, w.nsamp), dtype=torch.uint16 if w.input_bits == 16 else torch.uint8, pin_memory=True)
        x = t.numpy()
        datagen.generate(w.seed, w.nchans, w.nsamp, pl, dl, out=x, **w.gen_kw)
        return x, t
    return datagen.generate(w.seed, w.nchans, w.nsamp, pl, dl, **w.gen_kw), None


class OracleRun:
    """Oracle-side view of one workload: delay constants and binned chunks (cached per (chunk, bin))."""

    def __init__(self, w, x, per_width: bool = False):
        self.w, self.x, self.per_width = w, x, per_width
        self.k = oracle.delay_constants(w.freqs_mhz, w.tsamp_s)
        self._xb = {}

    def binned(self, start, length, b):
        key = (start, length, b)
        if key not in self._xb:
            self._xb = {k: v for k, v in self._xb.items() if k[:2] == (start, length)}   # keep one chunk's worth
            self._xb[key] = oracle.bin_time(self.x, start, length // b, b)
        return self._xb[key]

    def search(self, chunk, r_index, i0, i1, want=("D", "stats"), extra=0):
        start, length, n_out = chunk
        rng = self.w.ranges[r_index]
        xb = self.binned(start, length, rng[3])
        # the C ABI takes the threshold as float and widens it (include/aa.h): the oracle is handed the same double
        return oracle.search_rows(xb, self.k, rng, r_index, n_out // rng[3], self.w.widths, float(np.float32(self.w.threshold)), start,
                                  i0, i1, want=want, extra=extra, per_width=self.per_width)


def compare_candidates(got: np.ndarray, exp: np.ndarray, threshold: float, snr_rtol=1e-4, band=1e-3):
    """north_star 'Correctness': lists identical except for peaks within 1e-3 of the threshold; SNR within 1e-4 relative.
    Returns (n_matched, n_only_gpu_in_band, n_only_oracle_in_band); raises AssertionError otherwise."""
    def key(c):
        return list(zip(c["range"].tolist(), c["dm_index"].tolist(), c["sample"].tolist()))
    gk, ek = key(got), key(exp)
    gd = dict(zip(gk, range(len(gk))))
    ed = dict(zip(ek, range(len(ek))))
    assert len(gd) == len(gk), "duplicate candidates from the GPU"
    only_g = [k for k in gk if k not in ed]
    only_e = [k for k in ek if k not in gd]
    for k in only_g:
        assert abs(float(got["snr"][gd[k]]) - threshold) <= band, f"GPU-only candidate {k} snr={got['snr'][gd[k]]}"
    for k in only_e:
        assert abs(float(exp["snr"][ed[k]]) - threshold) <= band, f"oracle-only candidate {k} snr={exp['snr'][ed[k]]}"
    n = 0
    for k in gk:
        if k in ed:
            a, b = got[gd[k]], exp[ed[k]]
            assert abs(float(a["snr"]) - float(b["snr"])) <= snr_rtol * abs(float(b["snr"])), (k, a, b)
            assert int(a["width"]) == int(b["width"]) and float(a["dm"]) == float(b["dm"]), (k, a, b)
            n += 1
    return n, len(only_g), len(only_e)


def row_moments_from_input(x: np.ndarray, k: np.ndarray, rng, start: int, length: int, T: int, chan_block: int = 64):
    """SURVEY §8(c) pin (v), an O(C)-per-row route to sum_t D[i][t] and sum_t t*D[i][t] for EVERY row of a range that
    never forms D: per-channel prefix sums P, Q of the binned input and the oracle's delay table.
    Returns two int64 arrays [ndms]; arithmetic is modulo 2^64 (numpy int64 wraps), as on the device."""
    b = rng[3]
    dl = oracle.delay_table(k, rng)                         # [ndms][C]
    nd, C = dl.shape
    m0 = np.zeros(nd, np.int64)
    m1 = np.zeros(nd, np.int64)
    nb = length // b
    tt = np.arange(nb, dtype=np.int64)
    with np.errstate(over="ignore"):
        for c0 in range(0, C, chan_block):
            c1 = min(C, c0 + chan_block)
            xb = oracle.bin_time(x[c0:c1], start, nb, b).astype(np.int64)
            P = np.zeros((c1 - c0, nb + 1), np.int64)
            Q = np.zeros((c1 - c0, nb + 1), np.int64)
            np.cumsum(xb, axis=1, out=P[:, 1:])
            np.cumsum(xb * tt, axis=1, out=Q[:, 1:])
            d = dl[:, c0:c1]                                # [ndms][cb]
            ch = np.arange(c1 - c0)[None, :]
            dP = P[ch, d + T] - P[ch, d]
            dQ = Q[ch, d + T] - Q[ch, d]
            m0 += dP.sum(axis=1)
            m1 += (dQ - d * dP).sum(axis=1)
    return m0, m1


def row_moments_all_ranges(x: np.ndarray, k: np.ndarray, ranges, start: int, length: int, n_out: int, chan_block: int = 32,
                           threads: int | None = None):
    """The same identity as row_moments_from_input for EVERY row of EVERY range of a full-size chunk: the per-channel
    prefix sums P, Q are formed once per time-binning factor and shared by the ranges that use it; channel blocks run on
    a thread pool (numpy releases the GIL in cumsum). Returns [(m0, m1)] per range, int64 modulo 2^64."""
    import os
    from concurrent.futures import ThreadPoolExecutor
    C = x.shape[0]
    by_bin = {}
    for r, rng in enumerate(ranges):
        by_bin.setdefault(rng[3], []).append(r)
    tables = {r: oracle.delay_table(k, rng) for r, rng in enumerate(ranges)}
    out = {r: [np.zeros(rng[2], np.int64), np.zeros(rng[2], np.int64)] for r, rng in enumerate(ranges)}

    def block(b, c0):
        c1 = min(C, c0 + chan_block)
        nb = length // b
        xb = oracle.bin_time(x[c0:c1], start, nb, b)
        # P[n] = sum_{t<n} x[t]; the first-moment prefix Q[n] = sum_{t<n} t x[t] is n P[n] - R[n] with R[n] = sum_{m<=n} P[m]
        # (sum_{m=1..n} P[m] = sum_{t<n} (n - t) x[t]), so two cumulative sums serve both moments and Q is only formed at the
        # gathered indices. int64 modulo 2^64 throughout, like the GPU's sums.
        P = np.zeros((c1 - c0, nb + 1), np.int64)
        np.cumsum(xb, axis=1, dtype=np.int64, out=P[:, 1:])
        R = np.cumsum(P, axis=1)
        ch = np.arange(c1 - c0)[None, :]
        res = {}
        with np.errstate(over="ignore"):
            for r in by_bin[b]:
                T = n_out // b
                d = tables[r][:, c0:c1]
                P1, P0 = P[ch, d + T], P[ch, d]
                dP = P1 - P0
                dQ = ((d + T) * P1 - R[ch, d + T]) - (d * P0 - R[ch, d])
                res[r] = (dP.sum(axis=1), (dQ - d * dP).sum(axis=1))
        return res

    jobs = [(b, c0) for b in sorted(by_bin) for c0 in range(0, C, chan_block)]
    with ThreadPoolExecutor(max_workers=threads or min(16, os.cpu_count() or 1)) as ex:
        for res in ex.map(lambda j: block(*j), jobs):
            with np.errstate(over="ignore"):
                for r, (a0, a1) in res.items():
                    out[r][0] += a0
                    out[r][1] += a1
    return [tuple(out[r]) for r in range(len(ranges))]


def sampled_outputs(x: np.ndarray, k: np.ndarray, rng, start: int, T: int, points):
    """D[i][t'] of single outputs, each computed on its own from the definition (reading C5): the oracle's delay row of
    DM i, the oracle's binning of just the b input samples each channel contributes, one sum over channels.
    points: iterable of (i, t'). Returns int64 array."""
    b = rng[3]
    C = x.shape[0]
    ch = np.arange(C)
    out = []
    for (i, t) in points:
        d = oracle.delay_table(k, rng, i, i + 1)[0]                 # [C] binned samples
        u = start + (t + d) * b                                     # first unbinned sample of each channel's bin
        acc = 0
        for j in range(b):
            acc += int(x[ch, u + j].astype(np.int64).sum())
        out.append(acc)
    return np.array(out, np.int64)


# ---------------------------------------------------------------------------------------- the whole oracle, in parallel
# SURVEY §8(c) "Verification coverage": "run the single-threaded oracle as independent processes over DM slices with one
# halo row each side". The oracle itself is untouched (orc_search_rows adds the halo rows on its own); this only hands
# disjoint row slices [i0, i1) of one chunk to a pool of processes and gathers what they return. The binned chunk
# (oracle.bin_time, once per binning factor) lives in shared memory so that every process reads the same arrays.
_POOL_XB = {}


def _pool_init(spec):
    from multiprocessing import shared_memory
    for b, (name, shape) in spec.items():
        shm = shared_memory.SharedMemory(name=name)
        _POOL_XB[b] = (shm, np.ndarray(shape, dtype=np.uint16, buffer=shm.buf))


def _pool_slice(task):
    """One slice: rows [i0, i1) of range r. Returns the statistics, a 128-bit hash of every D row (as int32 bytes: D < 2^23)
    and the slice's candidates."""
    import hashlib
    (k, rng, r, T, widths, threshold, chunk_start, i0, i1, extra) = task
    xb = _POOL_XB[rng[3]][1]
    res = oracle.search_rows(xb, k, rng, r, T, widths, threshold, chunk_start, i0, i1, want=("D", "stats"), extra=extra)
    hashes = [hashlib.blake2b(np.ascontiguousarray(res["D"][q], dtype=np.int32).tobytes(), digest_size=16).digest()
              for q in range(i1 - i0)]
    return r, i0, i1, res["stats"], hashes, res["cands"]


def row_hash(row: np.ndarray) -> bytes:
    import hashlib
    return hashlib.blake2b(np.ascontiguousarray(row, dtype=np.int32).tobytes(), digest_size=16).digest()


def oracle_slices(ranges, rows_per_unit_cost: int = 16, keep_every: int = 1):
    """Disjoint DM slices covering every row of every range; a binned range's rows are cheaper, so its slices are taller.
    keep_every = n keeps every n-th slice (a bounded sample of the same partition)."""
    out = []
    for r, rng in enumerate(ranges):
        step = rows_per_unit_cost * rng[3]
        for q, i0 in enumerate(range(0, rng[2], step)):
            if q % keep_every == 0:
                out.append((r, i0, min(rng[2], i0 + step)))
    return out


def run_oracle_slices(w, x, chunk, slices, processes: int | None = None, extra: int = 0, on_idle=None):
    """Runs oracle.search_rows for every (r, i0, i1) of `slices` on `chunk` = (start, length, n_out) in a pool of
    single-threaded processes. Returns {(r, i0, i1): (stats [n][2], hashes [n], cands)}. `on_idle` (if given) is called in
    the parent between results, so GPU-side work can proceed while the pool computes."""
    import multiprocessing as mp
    import os
    from multiprocessing import shared_memory
    start, length, n_out = chunk
    k = oracle.delay_constants(w.freqs_mhz, w.tsamp_s)
    shms, spec = [], {}
    try:
        for b in sorted({w.ranges[r][3] for (r, _, _) in slices}):
            shape = (x.shape[0], length // b)
            shm = shared_memory.SharedMemory(create=True, size=int(np.prod(shape)) * 2)
            shms.append(shm)
            oracle.bin_time(x, start, length // b, b, out=np.ndarray(shape, dtype=np.uint16, buffer=shm.buf))
            spec[b] = (shm.name, shape)
        thr = float(np.float32(w.threshold))
        tasks = [(k, w.ranges[r], r, n_out // w.ranges[r][3], tuple(w.widths), thr, start, i0, i1, extra) for (r, i0, i1) in slices]
        tasks.sort(key=lambda t: -(t[8] - t[7]) / t[1][3])           # longest first
        out = {}
        ctx = mp.get_context("spawn")                                # fresh interpreters: no CUDA state is inherited
        with ctx.Pool(processes or os.cpu_count() or 1, initializer=_pool_init, initargs=(spec,)) as pool:
            it = pool.imap_unordered(_pool_slice, tasks)
            pending = len(tasks)
            while pending:
                try:
                    r, i0, i1, st, hs, c = it.next(timeout=0.05 if on_idle else None)
                except mp.TimeoutError:
                    on_idle()
                    continue
                out[(r, i0, i1)] = (st, hs, c)
                pending -= 1
        return out
    finally:
        for shm in shms:
            shm.close()
            shm.unlink()


class GpuRun:
    """The CUDA path through the C-ABI binding for one workload (plan -> strategy -> chunk loop)."""

    def __init__(self, w, x, time_major: bool = False, boxcar_overlap: bool = False, per_width: bool = False, **strategy_kw):
        """x is always the channel-major array [nchans][nsamp] the oracle sees; with time_major=True the library is handed
        its transpose x_tm[t][c] (the plain definition of the corner turn) through a time-major plan."""
        import paper_1912_07704_b200 as aa
        self.aa, self.w = aa, w
        self.x = np.ascontiguousarray(x.T) if time_major else x
        self.plan = aa.Plan(w.freqs_mhz, w.tsamp_s, w.ranges, w.widths, w.threshold, time_major=time_major,
                            boxcar_overlap=boxcar_overlap, per_width_stats=per_width, input_bits=w.input_bits,
                            input_max=w.max_value if w.input_bits == 16 else 0)
        self.extra = max(w.widths) - 1 if boxcar_overlap else 0          # reading C3x
        self.st = aa.Strategy(self.plan, x.shape[1], **strategy_kw)
        self.h = self.st.handle
        self.info = self.st.info
        self.chunks = [aa.aa_strategy_get_chunk(self.h, j) for j in range(self.info["nchunks"])]

    def dedisperse(self):
        return self.aa.aa_run_dedispersion(self.h, self.x)

    def sps(self):
        return self.aa.aa_run_sps(self.h)

    def row(self, r, i):
        return self.aa.aa_get_dedispersed_row(self.h, r, i)

    def stats(self, r, i):
        return self.aa.aa_get_row_stats(self.h, r, i)

    def width_stats(self, r, i, iw):
        return self.aa.aa_get_row_width_stats(self.h, r, i, iw)

    def moments(self, r):
        return self.aa.aa_get_row_moments(self.h, r, self.w.ranges[r][2])

    def candidates(self, **kw):
        return self.aa.aa_get_candidates(self.h, **kw)

    def close(self):
        self.st.close()
        self.plan.close()


def band_rows(ndms: int, centres, half: int = 2):
    """Bands [i0, i1) of 2*half+1 adjacent DM rows around each centre, clipped to the range, deduplicated."""
    out = []
    for c in centres:
        i0 = max(0, min(ndms - (2 * half + 1), c - half))
        i1 = min(ndms, i0 + 2 * half + 1)
        if (i0, i1) not in out:
            out.append((i0, i1))
    return out


def check_band(gpu: GpuRun, orc: OracleRun, chunk, r, i0, i1, *, after_sps: bool, cands=None):
    """Bit-exact D rows [i0,i1) and (after SPS) mu/sigma of the same rows; returns the oracle's candidates in the band's
    INTERIOR rows (those whose 3x3 neighbourhood lies inside the band or at the range edge)."""
    res = orc.search(chunk, r, i0, i1, want=("D", "stats"), extra=getattr(gpu, "extra", 0))
    for i in range(i0, i1):
        got = gpu.row(r, i)
        exp = res["D"][i - i0]
        assert got.shape == exp.shape, (r, i, got.shape, exp.shape)
        if not np.array_equal(got.astype(np.int64), exp):
            bad = np.flatnonzero(got.astype(np.int64) != exp)
            raise AssertionError(f"D mismatch range {r} row {i}: {len(bad)} samples, first at t={bad[:5]}, "
                                 f"got {got[bad[:5]]}, expected {exp[bad[:5]]}")
        if after_sps:
            mu, sg, n, it = gpu.stats(r, i)
            emu, esg = res["stats"][i - i0]
            assert mu == emu and sg == esg, (r, i, mu, emu, sg, esg)
    return res["cands"]


def check_bands(gpu: GpuRun, orc: OracleRun, chunk, bands, *, after_sps: bool, threads: int | None = None):
    """check_band for a list of bands [(r, i0, i1)] of one chunk. The oracle side (single-threaded C per call; ctypes releases the
    GIL) runs the bands on a thread pool over the host cores, the comparison with the CUDA path stays on the calling thread.
    Returns the oracle's candidates per band, in the order of `bands`."""
    import os
    from concurrent.futures import ThreadPoolExecutor
    start, length, n_out = chunk
    for b in sorted({orc.w.ranges[r][3] for (r, _, _) in bands}):
        orc.binned(start, length, b)                       # bin once, on this thread (the cache is not thread-safe)
    extra = getattr(gpu, "extra", 0)
    with ThreadPoolExecutor(max_workers=threads or min(16, os.cpu_count() or 1)) as ex:
        results = list(ex.map(lambda bd: orc.search(chunk, bd[0], bd[1], bd[2], want=("D", "stats"), extra=extra), bands))
    out = []
    for (r, i0, i1), res in zip(bands, results):
        for i in range(i0, i1):
            got = gpu.row(r, i)
            exp = res["D"][i - i0]
            assert got.shape == exp.shape, (r, i, got.shape, exp.shape)
            if not np.array_equal(got.astype(np.int64), exp):
                bad = np.flatnonzero(got.astype(np.int64) != exp)
                raise AssertionError(f"D mismatch range {r} row {i}: {len(bad)} samples, first at t={bad[:5]}, "
                                     f"got {got[bad[:5]]}, expected {exp[bad[:5]]}")
            if after_sps:
                mu, sg, n, it = gpu.stats(r, i)
                emu, esg = res["stats"][i - i0]
                assert mu == emu and sg == esg, (r, i, mu, emu, sg, esg)
        out.append(res["cands"])
    return out
