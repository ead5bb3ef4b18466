"""GPU parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times (the strategy's own tiling and
chunking): Mid (configs[1]), SKA-like (configs[2], the headline workload: against the WHOLE oracle, run in parallel over
DM slices), Low-frequency (configs[3]) and Streaming (configs[4]). Where the full oracle would take hours (Mid on one
core, Low-frequency, Streaming), SURVEY §8(c) "Verification coverage" applies:
  1. EVERY row of every range: sum_t D and sum_t t*D equal the values derived from the input's prefix sums (exact, int64);
  2. sampled single outputs D[i][t'], each computed on its own from the definition (random points + the corners of
     every range + tile-boundary columns), bit-exact;
  3. bands of 5 adjacent DM rows (first / middle / last of each range, plus the rows of injected pulses): bit-exact D,
     identical mu/sigma, identical candidates.
"""
import os

import numpy as np
import pytest

import datagen

from helpers import (GpuRun, OracleRun, band_rows, check_band, check_bands, compare_candidates, make_input, row_moments_all_ranges,
                     sampled_outputs)

pytestmark = pytest.mark.gpu


def _points(rng_np, ndms, T, n):
    pts = [(0, 0), (0, T - 1), (ndms - 1, 0), (ndms - 1, T - 1)]
    for t in (1023, 1024, 1025, T - 1024, (T // 1024) * 1024 - 1, (T // 1024) * 1024):      # K2 time-tile edges
        if 0 <= t < T:
            pts.append((int(rng_np.integers(0, ndms)), int(t)))
    for i in (31, 32, ndms - 33, (ndms // 32) * 32 - 1, (ndms // 32) * 32):                 # K2 DM-tile edges
        if 0 <= i < ndms:
            pts.append((int(i), int(rng_np.integers(0, T))))
    while len(pts) < n:
        pts.append((int(rng_np.integers(0, ndms)), int(rng_np.integers(0, T))))
    return pts


def _fullsize(name, points_per_range, pulse_bands):
    w = datagen.get_workload(name)
    x, pinned = make_input(w, pinned=True)
    before = datagen.checksum(x)
    gpu, orc = GpuRun(w, x, max_candidates=1 << 22), OracleRun(w, x)
    try:
        assert gpu.info["nchunks"] == 1
        chunk = gpu.chunks[0]
        start, length, n_out = chunk
        gpu.dedisperse()
        # 1. every row, two exact moments
        exp = row_moments_all_ranges(x, orc.k, w.ranges, start, length, n_out)
        for r, rng in enumerate(w.ranges):
            m0, m1 = gpu.moments(r)
            bad = np.flatnonzero((m0 != exp[r][0]) | (m1 != exp[r][1]))
            assert bad.size == 0, f"{name} range {r}: moment identity fails on rows {bad[:10]} ({bad.size} rows)"
        # 2. sampled outputs, one by one
        rs = np.random.default_rng(w.seed)
        for r, rng in enumerate(w.ranges):
            T = n_out // rng[3]
            pts = _points(rs, rng[2], T, points_per_range)
            want = sampled_outputs(x, orc.k, rng, start, T, pts)
            rows = {}
            for (i, t), e in zip(pts, want):
                if i not in rows:
                    rows[i] = gpu.row(r, i)
                assert int(rows[i][t]) == int(e), f"{name} range {r} D[{i}][{t}] = {int(rows[i][t])}, definition gives {int(e)}"
        # 3. bands with statistics and candidates
        gpu.sps()
        got = gpu.candidates(allow_overflow=False)
        pl, dms, _ = w.pulses()
        bands = []
        for r, rng in enumerate(w.ranges):
            centres = [0, rng[2] // 2, rng[2] - 1]
            hi = rng[0] + rng[1] * rng[2]
            centres += [int(round((d - rng[0]) / rng[1])) for d in dms[:pulse_bands] if rng[0] <= d < hi]
            bands += [(r, i0, i1) for (i0, i1) in band_rows(rng[2], [min(rng[2] - 1, max(0, c)) for c in centres])]
        for (r, i0, i1), e in zip(bands, check_bands(gpu, orc, chunk, bands, after_sps=True)):     # the oracle's bands run in parallel
            sel = (got["range"] == r) & (got["dm_index"] >= i0) & (got["dm_index"] < i1)
            compare_candidates(got[sel], e, w.threshold)
        nb = len(bands)
        assert datagen.checksum(x) == before          # the user's input is never written
        return gpu.info, len(got), nb
    finally:
        gpu.close()


def test_mid_full_size():
    info, ncand, nb = _fullsize("mid", points_per_range=400, pulse_bands=6)
    assert (info["overlap"], info["n_out"]) == (7243, 254901) and nb >= 3 and ncand > 0


def test_ska_full_size_whole_oracle():
    """BASELINE.json configs[2] (the headline workload) at full size against the WHOLE oracle (SURVEY §8(c) "Verification
    coverage": "SKA-like - full if the GPU box has >= 16 cores"): the single-threaded oracle runs as independent processes
    over DM slices with one halo row each side (helpers.run_oracle_slices); compared are EVERY element of D of all 5 150
    rows (128-bit hash of each int32 row on both sides), mu and sigma of every row with ==, and the whole candidate list.
    Fraction that runs: all slices when the box has >= 12 cores (or AA_TEST_SKA_ORACLE_EVERY=1); on a smaller box every
    n-th slice (n = 16 // cores, at least 2) of the same partition, and the remaining rows get the all-rows moment
    identity instead. The docstring of oracle_slices states the partition."""
    from helpers import oracle_slices, row_hash, run_oracle_slices
    w = datagen.get_workload("ska")
    x, _ = make_input(w)                                  # pageable: the oracle processes map their own shared copies
    before = datagen.checksum(x)
    cores = os.cpu_count() or 1
    every = int(os.environ.get("AA_TEST_SKA_ORACLE_EVERY", "0")) or (1 if cores >= 12 else max(2, 16 // cores))
    gpu = GpuRun(w, x, max_candidates=1 << 22)
    try:
        assert gpu.info["nchunks"] == 1
        assert (gpu.info["overlap"], gpu.info["n_out"], gpu.info["max_bin"]) == (32384, 491904, 8)
        chunk = gpu.chunks[0]
        start, length, n_out = chunk
        gpu.dedisperse()
        gpu.sps()
        got = gpu.candidates(allow_overflow=False)
        slices = oracle_slices(w.ranges, rows_per_unit_cost=16, keep_every=every)
        # GPU side, gathered while the pool computes: hash of every D row and its statistics
        todo = [(r, i) for (r, i0, i1) in slices for i in range(i0, i1)]
        gh, gs = {}, {}

        def on_idle(n=64):
            for _ in range(min(n, len(todo))):
                r, i = todo.pop()
                gh[(r, i)] = row_hash(gpu.row(r, i))
                gs[(r, i)] = gpu.stats(r, i)[:2]

        res = run_oracle_slices(w, x, chunk, slices, on_idle=on_idle)
        while todo:
            on_idle()
        nrows, exp = 0, []
        for (r, i0, i1) in slices:
            st, hs, c = res[(r, i0, i1)]
            for i in range(i0, i1):
                assert gh[(r, i)] == hs[i - i0], f"ska range {r} row {i}: D differs from the oracle"
                assert gs[(r, i)] == (st[i - i0][0], st[i - i0][1]), (r, i, gs[(r, i)], tuple(st[i - i0]))
                nrows += 1
            exp.append(c)
        exp = np.concatenate(exp)
        if every == 1:
            assert nrows == w.ndms_total == 5150
            n, og, oe = compare_candidates(got, exp, w.threshold)
            assert n + og == len(got) and n + oe == len(exp) and len(got) > 1000
        else:
            sel = np.zeros(len(got), bool)
            for (r, i0, i1) in slices:
                sel |= (got["range"] == r) & (got["dm_index"] >= i0) & (got["dm_index"] < i1)
            compare_candidates(got[sel], exp, w.threshold)
            orc = OracleRun(w, x)
            em = row_moments_all_ranges(x, orc.k, w.ranges, start, length, n_out)
            for r in range(len(w.ranges)):
                m0, m1 = gpu.moments(r)
                assert np.array_equal(m0, em[r][0]) and np.array_equal(m1, em[r][1]), r
        assert datagen.checksum(x) == before          # the user's input is never written
    finally:
        gpu.close()


def test_ska16_full_size():
    """The SKA-like configuration delivered as 16-bit samples of 12-bit depth (PAPER.md:47 step 1) at full size:
    offset-uint8 forms at bin 1/2/4 on 4096 channels, the offset-uint16 kernel on the bin-8 range, the 4.29 GB chunk through
    the 3-group copy. All-row moments, sampled outputs and bands; the pulses are the ska workload's (same seed), so the list
    has the same length as the 8-bit run's."""
    info, ncand, nb = _fullsize("ska16", points_per_range=60, pulse_bands=1)
    assert info["input_bits"] == 16 and info["input_max"] == 4095 and nb >= 15 and ncand > 0


def test_lowf_full_size():
    """BASELINE.json configs[3] at full size (4096 channels x 2^21 samples, 6000 DM trials, delays up to 545 316 samples):
    all-row moments, sampled outputs and bands (first / middle / last of each range + one pulse band)."""
    info, ncand, nb = _fullsize("lowf", points_per_range=60, pulse_bands=1)
    assert (info["overlap"], info["n_out"], info["max_bin"]) == (545316, 1551836, 4) and nb >= 9 and ncand > 0


def test_stream_full_size_selected_chunks():
    """BASELINE.json configs[4] at full size (600 s, 40 GB budget, double-buffered H2D): the whole chunk loop runs; EVERY chunk
    gets the all-row moment identity ("every row of every chunk"; the oracle side of chunk j runs on a worker thread
    while the GPU works on the chunks after it); the first, a middle and the last (short) chunk also get sampled outputs and one
    band per range, and the candidate lists of those bands are compared; status codes are checked on every chunk."""
    from concurrent.futures import ThreadPoolExecutor
    w = datagen.get_workload("stream")
    x, pinned = make_input(w, pinned=True)
    gpu, orc = GpuRun(w, x, budget_bytes=w.budget_bytes, max_candidates=1 << 23), OracleRun(w, x)
    try:
        n = gpu.info["nchunks"]
        assert n >= 10 and gpu.info["arena_bytes_used"] <= w.budget_bytes
        check = {0, n // 2, n - 1}
        rs = np.random.default_rng(w.seed)
        exp_bands = []
        pool, pending = ThreadPoolExecutor(max_workers=1), []
        for j, chunk in enumerate(gpu.chunks):
            start, length, n_out = chunk
            gpu.dedisperse()
            if j not in check:                    # all-row moments of this chunk: GPU sums now (D is overwritten by the next chunk),
                got_m = [gpu.moments(r) for r in range(len(w.ranges))]            # the oracle's side in the background
                pending.append((j, got_m, pool.submit(row_moments_all_ranges, x[:, start:start + length], orc.k, w.ranges, 0, length,
                                                      n_out, 32, None)))
            if j in check:
                exp = row_moments_all_ranges(x[:, start:start + length], orc.k, w.ranges, 0, length, n_out)
                for r, rng in enumerate(w.ranges):
                    m0, m1 = gpu.moments(r)
                    assert np.array_equal(m0, exp[r][0]) and np.array_equal(m1, exp[r][1]), (j, r)
                    T = n_out // rng[3]
                    pts = _points(rs, rng[2], T, 24)
                    want = sampled_outputs(x, orc.k, rng, start, T, pts)
                    rows = {}
                    for (i, t), e in zip(pts, want):
                        if i not in rows:
                            rows[i] = gpu.row(r, i)
                        assert int(rows[i][t]) == int(e), (j, r, i, t)
            status = gpu.sps()
            assert status == (gpu.aa.AA_STATUS_FINISHED if j == n - 1 else gpu.aa.AA_STATUS_CHUNK_DONE)
            if j in check:
                bands = [(r,) + band_rows(rng[2], [rng[2] // 2])[0] for r, rng in enumerate(w.ranges)]
                for (r, i0, i1), e in zip(bands, check_bands(gpu, orc, chunk, bands, after_sps=True)):
                    exp_bands.append((r, i0, i1, start, n_out, e))
        got = gpu.candidates()
        for (r, i0, i1, start, n_out, e) in exp_bands:
            sel = (got["range"] == r) & (got["dm_index"] >= i0) & (got["dm_index"] < i1) & (got["sample"] >= start) & (got["sample"] < start + n_out)
            compare_candidates(got[sel], e, w.threshold)
        assert len(got) > 0
        assert len(pending) + len(check) == n
        for (j, got_m, fut) in pending:
            exp = fut.result()
            for r in range(len(w.ranges)):
                assert np.array_equal(got_m[r][0], exp[r][0]) and np.array_equal(got_m[r][1], exp[r][1]), (j, r)
        pool.shutdown()
    finally:
        gpu.close()
