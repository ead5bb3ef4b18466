"""GPU parity tests proper (-m gpu): the CUDA path, called through the C-ABI binding, against the oracle on the same
seeded bytes. Bars (BASELINE.json north_star "Correctness"): dedispersed sums bit-exact; mu/sigma/SNR taken in IEEE
double on both sides (so they are compared exactly, far inside the stated 1e-4); candidate lists identical except peaks
within 1e-3 of the threshold.

Coverage (SURVEY §8(c) "Verification coverage"): small configs — every row; larger ones — (1) the all-rows moment identity
sum_t D, sum_t t*D computed from the INPUT's prefix sums for every row of every range, (2) bit-exact D, statistics and
candidates on bands of adjacent DM rows (first / middle / last of each range and around injected pulses).
"""
import numpy as np
import pytest

import datagen
from datagen.workloads import Workload, scaled

from helpers import GpuRun, OracleRun, band_rows, check_band, check_bands, compare_candidates, make_input, row_moments_from_input

pytestmark = pytest.mark.gpu


def _full_parity(w, x, **kw):
    """Every row of every range of every chunk: D, statistics, candidates."""
    gpu, orc = GpuRun(w, x, **kw), OracleRun(w, x, per_width=kw.get("per_width", False))
    try:
        exp_all = []
        for j, chunk in enumerate(gpu.chunks):
            gpu.dedisperse()
            status = gpu.sps()
            assert status == (gpu.aa.AA_STATUS_FINISHED if j == len(gpu.chunks) - 1 else gpu.aa.AA_STATUS_CHUNK_DONE)
            for r, rng in enumerate(w.ranges):
                exp_all.append(check_band(gpu, orc, chunk, r, 0, rng[2], after_sps=True))
        got = gpu.candidates()
        exp = np.concatenate(exp_all) if exp_all else got[:0]
        stats = compare_candidates(got, exp, w.threshold)
        return gpu.info, got, exp, stats
    finally:
        gpu.close()


def _band_parity(w, x, centres_per_range, **kw):
    """All-rows moment identity + bands. centres_per_range: {range: [dm_index, ...]}."""
    gpu, orc = GpuRun(w, x, **kw), OracleRun(w, x)
    try:
        ncheck = 0
        for j, chunk in enumerate(gpu.chunks):
            gpu.dedisperse()
            start, length, n_out = chunk
            for r, rng in enumerate(w.ranges):
                m0, m1 = gpu.moments(r)
                e0, e1 = row_moments_from_input(x, orc.k, rng, start, length, n_out // rng[3])
                bad = np.flatnonzero((m0 != e0) | (m1 != e1))
                assert bad.size == 0, f"chunk {j} range {r}: moment identity fails on rows {bad[:10]} ({bad.size} rows)"
            gpu.sps()
            got = gpu.candidates()
            bands = [(r, i0, i1) for r, rng in enumerate(w.ranges)
                     for (i0, i1) in band_rows(rng[2], centres_per_range.get(r, [0, rng[2] // 2, rng[2] - 1]))]
            for (r, i0, i1), exp in zip(bands, check_bands(gpu, orc, chunk, bands, after_sps=True)):
                sel = (got["range"] == r) & (got["dm_index"] >= i0) & (got["dm_index"] < i1) & \
                      (got["sample"] >= start) & (got["sample"] < start + n_out)
                compare_candidates(got[sel], exp, w.threshold)
                ncheck += 1
        return gpu.info, ncheck
    finally:
        gpu.close()


# ------------------------------------------------------------------------------------------------ Tiny (config 0)
def test_tiny_every_row_and_candidates():
    w = datagen.get_workload("tiny")
    x, _ = make_input(w)
    before = datagen.checksum(x)
    info, got, exp, (nmatch, og, oe) = _full_parity(w, x)
    assert datagen.checksum(x) == before                      # the API may not modify the user's input
    assert (info["overlap"], info["n_out"], info["nchunks"]) == (65, 8127, 1)
    assert nmatch == len(exp) and og == 0 and oe == 0 and len(got) > 0
    top = got[np.argmax(got["snr"])]
    # BASELINE.json config "Tiny": the injected pulse (DM 50, t0 3000, width 4) must be recovered within one sample
    assert abs(int(top["dm_index"]) - 50) <= 1 and abs(int(top["sample"]) - 3000) <= 1 and int(top["width"]) == 4


# ------------------------------------------------------------------------------------------------ ragged / degenerate shapes
@pytest.mark.parametrize("nchans,nsamp,ranges", [
    (61, 5003, ((0.0, 1.3, 37, 1), (48.1, 2.6, 5, 2), (61.1, 5.0, 33, 4), (226.1, 9.0, 3, 8))),   # nothing a multiple of a tile
    (1, 2100, ((0.0, 1.0, 3, 1),)),                                                                  # one channel: D == x
    (8, 1500, ((0.0, 50.0, 1, 1), (50.0, 10.0, 2, 8))),                                              # single-row ranges
    (300, 9000, ((0.0, 0.5, 65, 2),)),                                                               # > 256/bin channels: 16-bit carries
])
def test_ragged_shapes_every_row(nchans, nsamp, ranges):
    w = Workload("ragged", nchans, 420.0, -100.0 / max(nchans, 2), 2048e-6, nsamp, ranges, (1, 2, 3, 7, 16), 5.0,
                 seed=77 + nchans, npulses=3, pulse_dm=(5.0, 60.0), pulse_width_max=8, pulse_snr=(10.0, 25.0))
    x, _ = make_input(w)
    info, got, exp, (nmatch, og, oe) = _full_parity(w, x)
    assert nmatch + og == len(got) and nmatch + oe == len(exp)


def test_extreme_input_values_do_not_overflow_packed_lanes():
    """All-255 and all-0 inputs: the packed 8/16-bit lanes of K2 must carry exactly (closed form D = C*b*v)."""
    for v in (255, 0):
        w = Workload("const", 1024, 1500.0, -0.25, 64e-6, 6000, ((0.0, 2.0, 40, 1), (80.0, 4.0, 33, 8)), (1, 4), 6.0,
                     seed=1, npulses=0, pulse_dm=(0.0, 0.0), pulse_width_max=1)
        x = np.full((w.nchans, w.nsamp), v, np.uint8)
        gpu = GpuRun(w, x)
        try:
            gpu.dedisperse()
            for r, rng in enumerate(w.ranges):
                for i in (0, rng[2] // 2, rng[2] - 1):
                    assert np.all(gpu.row(r, i) == w.nchans * rng[3] * v)
            gpu.sps()
            assert len(gpu.candidates()) == 0                 # constant rows: sigma == 0, no candidates
        finally:
            gpu.close()


# ------------------------------------------------------------------------------------------------ Mid / SKA-like shapes, shortened
def test_mid_shape_bands_and_all_row_moments():
    w = scaled(datagen.get_workload("mid"), nsamp=48_000, name="mid48k")
    x, _ = make_input(w)
    pl, dms, _ = w.pulses()
    centres = sorted({0, 500, 1000} | {int(round(d / 0.5)) for d in dms[:4]})
    info, n = _band_parity(w, x, {0: centres})
    assert info["overlap"] == 7243 and n >= 3


def test_ska_shape_bands_and_all_row_moments():
    w = scaled(datagen.get_workload("ska"), nsamp=72_000, name="ska72k")
    x, _ = make_input(w)
    info, n = _band_parity(w, x, {})
    assert info["overlap"] == 32384 and info["max_bin"] == 8 and n == 15


def test_lowf_shape_wide_windows():
    """Low-frequency band: delay grows ~54 samples per DM step at the bottom channel (wide per-tile windows)."""
    lw = datagen.get_workload("lowf")
    w = scaled(lw, nsamp=620_000, name="lowf620k", nchans=4096,
               ranges=((0.0, 0.05, 70, 1), (100.0, 0.1, 40, 2), (490.0, 0.1, 100, 4)))
    x, _ = make_input(w)
    info, n = _band_parity(w, x, {})
    assert n == 9


# ------------------------------------------------------------------------------------------------ chunked (streaming) path
def test_chunked_run_matches_oracle_per_chunk_and_is_chunk_invariant():
    w = scaled(datagen.get_workload("mid"), nsamp=40_000, name="mid40k", ranges=((0.0, 0.5, 201, 1), (100.0, 1.0, 64, 2)))
    x, pinned = make_input(w, pinned=True)
    info, got, exp, (nmatch, og, oe) = _full_parity(w, x, chunk_len_hint=9_000)
    assert info["nchunks"] >= 4 and info["overlap"] % 2 == 0
    assert nmatch + og == len(got) and nmatch + oe == len(exp)
    # chunk invariance of D: the single-chunk run equals the concatenation of the chunked run
    one = GpuRun(w, x)
    many = GpuRun(w, x, chunk_len_hint=9_000)
    try:
        one.dedisperse()
        rows = {(0, 0): [], (0, 200): [], (1, 63): []}
        for _ in many.chunks:
            many.dedisperse()
            for key in rows:
                rows[key].append(many.row(*key))
            many.sps()
        for (r, i), parts in rows.items():
            cat = np.concatenate(parts)
            assert np.array_equal(cat, one.row(r, i)[:len(cat)])
    finally:
        one.close()
        many.close()


# ------------------------------------------------------------------------------------------------ replicas over chunks (N > 1 path)
def test_sharded_strategies_match_the_oracle_per_shard_and_reproduce_the_single_run():
    """rank r of W owns chunks r, r+W, ...; no exchange. Two sharded strategies (run one after
    the other on this one GPU, each with its own arena, as two ranks would): every chunk a shard owns is compared with the
    ORACLE (every D row bit-exact, every mu/sigma, the shard's candidate list), which also exercises the shard's
    double-buffer parity ((j / world) & 1); together the shards give exactly the unsharded list."""
    from paper_1912_07704_b200 import replicas
    w = scaled(datagen.get_workload("mid"), nsamp=40_000, name="mid40k", ranges=((0.0, 0.5, 120, 1), (60.0, 1.0, 40, 2)))
    x, pinned = make_input(w, pinned=True)
    one = GpuRun(w, x, chunk_len_hint=9_000)
    try:
        ref = one.st.run(x)
        nchunks, n_out = one.info["nchunks"], one.info["n_out"]
    finally:
        one.close()
    assert nchunks >= 4 and len(ref) > 0
    orc = OracleRun(w, x)
    parts, owned = [], []
    for rank in range(2):
        g = GpuRun(w, x, chunk_len_hint=9_000)
        try:
            g.st.shard(rank, 2)
            assert g.st.info["next_chunk"] == rank
            mine = replicas.chunks_of_rank(nchunks, rank, 2)
            exp_all = []
            for n, j in enumerate(mine):
                assert g.aa.aa_strategy_get_info(g.h)["next_chunk"] == j
                g.dedisperse()                                   # the shard's cursor: chunks rank, rank + 2, ...
                status = g.sps()
                assert status == (g.aa.AA_STATUS_FINISHED if n == len(mine) - 1 else g.aa.AA_STATUS_CHUNK_DONE)
                for r, rng in enumerate(w.ranges):
                    exp_all.append(check_band(g, orc, g.chunks[j], r, 0, rng[2], after_sps=True))
            c = g.candidates()
            nm, og, oe = compare_candidates(c, np.concatenate(exp_all), w.threshold)
            assert nm + og == len(c) and nm + oe == sum(len(e) for e in exp_all)
            assert set((c["sample"] // n_out).tolist()) <= set(mine)
            # and the one-call loop of the same shard gives the same list
            g.st.shard(rank, 2)
            c2 = g.st.run(x)
            assert np.array_equal(c2, c)
            parts.append(c)
            owned += mine
        finally:
            g.close()
    assert sorted(owned) == list(range(nchunks))
    merged = replicas.canonical_order(np.concatenate(parts), n_out)
    assert len(merged) == len(ref)
    for f in ref.dtype.names:
        assert np.array_equal(merged[f], ref[f]), f


# ------------------------------------------------------------------------------------------------ reading C9 on the GPU
def test_candidate_record_in_binned_ranges_and_later_chunks_gpu():
    """GPU twin of tests/test_oracle_pins.py::test_candidate_record_in_binned_ranges_and_later_chunks: pulses injected at
    known UNBINNED samples in a bin-4 range and in chunks 1 and 2 come back at those coordinates through the C ABI
    (sample = chunk_start + bin*t', width = bin*w*), and the whole run equals the oracle."""
    base = datagen.get_workload("tiny")
    w = scaled(base, name="tiny_c9", nsamp=16384, ranges=((0.0, 1.0, 40, 1), (40.0, 2.0, 30, 4)), widths=(1, 2, 4, 8, 16),
               fixed_pulses=((20.0, 5000, 4, 14.0), (70.0, 9000, 16, 8.0)))
    x, _ = make_input(w)
    info, got, exp, (nmatch, og, oe) = _full_parity(w, x, chunk_len_hint=4096)
    assert info["nchunks"] >= 4 and nmatch + og == len(got) and nmatch + oe == len(exp)
    for (r_index, t0, width, dm_index) in ((0, 5000, 4, 20), (1, 9000, 16, 15)):
        b = w.ranges[r_index][3]
        j = t0 // info["n_out"]
        sel = got[(got["range"] == r_index) & (got["sample"] // info["n_out"] == j)]
        top = sel[np.argmax(sel["snr"])]
        assert abs(int(top["dm_index"]) - dm_index) <= 1 and abs(int(top["sample"]) - t0) <= b
        assert int(top["width"]) % b == 0 and width // 2 <= int(top["width"]) <= 2 * width


def test_threshold_that_is_not_float_exact():
    """The library takes the threshold as float and widens it; the oracle is handed the same double (helpers.OracleRun).
    6.1 is not representable: with thousands of noise peaks near it, a double-vs-float mix-up would show as unmatched
    candidates outside the 1e-3 band only by luck, so the lists are also required to agree in LENGTH."""
    w = scaled(datagen.get_workload("tiny"), name="tiny_thr", threshold=6.1, widths=(1, 2, 4, 8, 16))
    x, _ = make_input(w)
    info, got, exp, (nmatch, og, oe) = _full_parity(w, x)
    assert len(got) == len(exp) and nmatch == len(exp) and len(got) > 0


# ------------------------------------------------------------------------------------------------ time-major input (corner turn)
@pytest.mark.parametrize("nchans,nsamp,ranges,hint", [
    (64, 8192, ((0.0, 1.0, 101, 1),), 0),                                              # Tiny, one chunk
    (61, 5003, ((0.0, 1.3, 37, 1), (48.1, 2.6, 5, 2), (226.1, 9.0, 3, 8)), 0),         # nothing a multiple of a tile or of 4
    (300, 30000, ((0.0, 0.5, 65, 2), (10.0, 0.5, 40, 1)), 8000),                       # several chunks: double-buffered staging
])
def test_time_major_input_gives_the_channel_major_result(nchans, nsamp, ranges, hint):
    """PAPER.md:47 step 1: telescopes deliver x[t][c]. The library corner-turns each chunk on the device; the oracle is
    handed the transpose (the plain definition). Every D row, every statistic and the candidate list must be identical."""
    w = Workload("tm", nchans, 1500.0, -100.0 / max(nchans, 2), 256e-6, nsamp, ranges, (1, 2, 4, 8), 5.5,
                 seed=4242 + nchans, npulses=3, pulse_dm=(5.0, 30.0), pulse_width_max=6, pulse_snr=(10.0, 25.0))
    x, _ = make_input(w)
    kw = dict(chunk_len_hint=hint) if hint else {}
    gpu, orc = GpuRun(w, x, time_major=True, **kw), OracleRun(w, x)
    try:
        assert gpu.info["input_layout"] == gpu.aa.AA_LAYOUT_TIME_MAJOR and gpu.x.shape == (nsamp, nchans)
        before = gpu.x.copy()
        exp_all = []
        for chunk in gpu.chunks:
            gpu.dedisperse()
            gpu.sps()
            for r, rng in enumerate(w.ranges):
                exp_all.append(check_band(gpu, orc, chunk, r, 0, rng[2], after_sps=True))
        got = gpu.candidates()
        n, og, oe = compare_candidates(got, np.concatenate(exp_all), w.threshold)
        assert n + og == len(got) and n + oe == sum(len(e) for e in exp_all)
        assert np.array_equal(gpu.x, before)
        if hint:
            assert gpu.info["nchunks"] >= 3
    finally:
        gpu.close()


def test_time_major_device_chunk_and_layout_errors():
    import torch
    aa = __import__("paper_1912_07704_b200")
    w = datagen.get_workload("tiny")
    x, _ = make_input(w)
    gpu, orc = GpuRun(w, x, time_major=True), OracleRun(w, x)
    try:
        xd = torch.from_numpy(gpu.x).cuda()                       # [nsamp][nchans] on the device
        aa.aa_run_dedispersion_device(gpu.h, xd, xd.stride(0))
        gpu.sps()
        exp = check_band(gpu, orc, gpu.chunks[0], 0, 0, w.ranges[0][2], after_sps=True)
        compare_candidates(gpu.candidates(), exp, w.threshold)
        aa.aa_strategy_reset(gpu.h)
        with pytest.raises(aa.AaError) as e:                      # stride shorter than a time row
            aa.aa_run_dedispersion(gpu.h, gpu.x, w.nchans - 1)
        assert e.value.status == aa.AA_ERR_INVALID_ARG and "nchans" in e.value.message
        with pytest.raises(aa.AaError) as e:
            aa.aa_plan_set_input_layout(gpu.plan.handle, 7)
        assert e.value.status == aa.AA_ERR_INVALID_ARG and "layout" in e.value.message
    finally:
        gpu.close()


# ------------------------------------------------------------------------------------------------ reading C7m (per-width measured statistics)
def _width_stats_parity(w, x, rows_per_range=6, **kw):
    """mu_w, sigma_w, p_w of every plan width on sampled rows, == the oracle's (reading C7m), on the current chunk(s)."""
    import oracle
    gpu, orc = GpuRun(w, x, per_width=True, **kw), OracleRun(w, x, per_width=True)
    n = 0
    try:
        for chunk in gpu.chunks:
            gpu.dedisperse()
            gpu.sps()
            start, length, n_out = chunk
            for r, rng in enumerate(w.ranges):
                T = n_out // rng[3]
                for i in sorted({int(q) for q in np.linspace(0, rng[2] - 1, rows_per_range)}):
                    row = gpu.row(r, i).astype(np.int64)                      # T + E samples (already checked bit-exact elsewhere)
                    _, _, ws = oracle.boxcar_snr_perwidth(row, T, w.widths)
                    for iw in range(len(w.widths)):
                        mu, sg, pv = gpu.width_stats(r, i, iw)
                        assert (mu, sg, float(pv)) == (ws[iw][0], ws[iw][1], ws[iw][2]), (r, i, iw, (mu, sg, pv), tuple(ws[iw]))
                        n += 1
        return n
    finally:
        gpu.close()


@pytest.mark.parametrize("kw", [{}, {"chunk_len_hint": 4096}, {"boxcar_overlap": True, "chunk_len_hint": 4096}])
def test_per_width_statistics_every_row_matches_the_oracle(kw):
    """SURVEY §8(f3) / DESIGN.md reading C7m with the option on: every row's D, every candidate (whole list) and the
    per-width statistics equal the oracle's, on a plan with binned ranges, widths that are not powers of two, several chunks
    and (third case) boxcars that cross the chunk end (reading C3x), where n_w differs per width."""
    w = scaled(datagen.get_workload("tiny"), name="tiny_pw", nsamp=16384, ranges=((0.0, 1.0, 40, 1), (40.0, 2.0, 30, 4), (100.0, 4.0, 9, 8)),
               widths=(1, 2, 3, 8, 21, 64), fixed_pulses=((20.0, 5000, 4, 14.0), (70.0, 9000, 16, 8.0)), threshold=5.5)
    x, _ = make_input(w)
    info, got, exp, (nmatch, og, oe) = _full_parity(w, x, per_width=True, **kw)
    assert nmatch + og == len(got) and nmatch + oe == len(exp) and len(got) > 10
    assert _width_stats_parity(w, x, **kw) > 0


def test_per_width_statistics_on_red_noise_differ_from_sqrt_w_scaling_and_match_the_oracle():
    """A slow baseline wander common to all channels makes every dedispersed row RED: sigma of a wide boxcar is then far
    above sqrt(w) sigma_1, reading C7 reports inflated SNRs for wide boxcars and reading C7m does not. Both runs must equal
    the oracle in their own reading; the C7m run must find fewer wide candidates than the C7 run on the same bytes."""
    base = scaled(datagen.get_workload("tiny"), name="tiny_red", nsamp=32768, ranges=((0.0, 1.0, 48, 1), (48.0, 2.0, 16, 2)),
                  widths=(1, 2, 4, 8, 16, 32, 64), fixed_pulses=((30.0, 9000, 8, 12.0),), threshold=6.0)
    x, _ = make_input(base)
    rs = np.random.default_rng(5)
    wander = np.cumsum(rs.normal(0.0, 0.35, base.nsamp))
    wander -= np.convolve(wander, np.ones(2048) / 2048, mode="same")            # keep it inside the byte range
    x = np.clip(np.round(x.astype(np.float64) + wander[None, :]), 0, 255).astype(np.uint8)
    _, got_w, exp_w, (nm_w, og_w, oe_w) = _full_parity(base, x, per_width=True)
    _, got_c, exp_c, (nm_c, og_c, oe_c) = _full_parity(base, x)
    assert nm_w + og_w == len(got_w) and nm_w + oe_w == len(exp_w)
    assert nm_c + og_c == len(got_c) and nm_c + oe_c == len(exp_c)
    wide_c = int(np.sum(got_c["width"] >= 32)); wide_w = int(np.sum(got_w["width"] >= 32))
    assert wide_c > 4 * max(1, wide_w), (wide_c, wide_w)
    assert _width_stats_parity(base, x, rows_per_range=4) > 0


def test_per_width_statistics_full_length_rows_and_degenerate_widths():
    """Rows of the Mid shape (T ~ 58 000: many tiles of K3w, ragged tail) with widths up to 512; a constant input gives
    sigma_w = 0 for every width (no SNR, no candidates) on both sides; the hook refuses plans without the option."""
    import paper_1912_07704_b200 as aa
    w = scaled(datagen.get_workload("mid"), name="mid_pw", nsamp=65_536, nchans=256, ranges=((0.0, 0.5, 24, 1), (12.0, 1.0, 10, 2)),
               widths=(1, 2, 4, 8, 16, 32, 64, 128, 256, 512), npulses=4, pulse_dm=(2.0, 20.0))
    x, _ = make_input(w)
    info, got, exp, (nmatch, og, oe) = _full_parity(w, x, per_width=True)
    assert nmatch + og == len(got) and nmatch + oe == len(exp)
    assert _width_stats_parity(w, x, rows_per_range=3) > 0
    flat = np.full_like(x, 100)
    info, got, exp, _ = _full_parity(w, flat, per_width=True)
    assert len(got) == 0 and len(exp) == 0
    g = GpuRun(w, x)
    try:
        g.dedisperse(); g.sps()
        with pytest.raises(aa.AaError) as e:
            g.width_stats(0, 0, 0)
        assert e.value.status == aa.AA_ERR_ORDER
    finally:
        g.close()
