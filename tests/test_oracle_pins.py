"""Pins of the oracle against things other than itself (-m "not gpu").

Each test names what fixes the expected value: a cited golden file, exact rational arithmetic, a closed form,
an invariant, a library routine the oracle does not use, or pure-Python brute force on a tiny input.
"""
from fractions import Fraction
from pathlib import Path

import numpy as np
import pytest

import datagen
import oracle

GOLD = Path(__file__).resolve().parent / "golden"


def _rows(name):
    for line in (GOLD / name).read_text().splitlines():
        line = line.strip()
        if line and not line.startswith("#"):
            yield line.split()


def _exact_delay(freqs, c, dm, tsamp, b):
    """north_star formula in exact rational arithmetic on the double-valued inputs; round half away from zero."""
    f, f0 = Fraction(float(freqs[c])), Fraction(float(freqs[0]))
    v = Fraction(4148808, 1000) * Fraction(float(dm)) * (1 / (f * f) - 1 / (f0 * f0)) / Fraction(float(tsamp)) / b
    q = int(v)            # v >= 0
    return q + (1 if v - q >= Fraction(1, 2) else 0), v


# ------------------------------------------------------------------------------------------------ C2 delays
def test_delay_golden_values():
    for wl, c, dm, b, exp in _rows("delays.txt"):
        w = datagen.get_workload(wl)
        k = oracle.delay_constants(w.freqs_mhz, w.tsamp_s)
        assert oracle.delay(k[int(c)], float(dm), int(b)) == int(exp), (wl, c, dm, b)
        assert _exact_delay(w.freqs_mhz, int(c), float(dm), w.tsamp_s, int(b))[0] == int(exp)


@pytest.mark.parametrize("wl", ["tiny", "mid", "ska", "lowf"])
def test_delay_matches_exact_rational_on_samples(wl):
    w = datagen.get_workload(wl)
    k = oracle.delay_constants(w.freqs_mhz, w.tsamp_s)
    rng = np.random.default_rng(11)
    for r in w.ranges:
        cs = np.concatenate([[0, 1, w.nchans - 1], rng.integers(0, w.nchans, 60)])
        js = np.concatenate([[0, 1, r[2] - 1], rng.integers(0, r[2], 60)])
        for c, i in zip(cs, js):
            dm = oracle.dm_value(r[0], r[1], int(i))
            exp, v = _exact_delay(w.freqs_mhz, int(c), dm, w.tsamp_s, r[3])
            got = oracle.delay(k[int(c)], dm, r[3])
            # double evaluation may differ from the exact value only within 1e-9 of a tie
            assert got == exp or abs((v - int(v)) - Fraction(1, 2)) < Fraction(1, 10**9), (wl, c, i)


def test_delay_zero_and_monotone():
    w = datagen.get_workload("ska")
    k = oracle.delay_constants(w.freqs_mhz, w.tsamp_s)
    assert k[0] == 0.0 and np.all(np.diff(k) > 0)
    for r in w.ranges:
        assert oracle.delay(k[0], r[0] + 5 * r[1], r[3]) == 0
        assert oracle.delay(k[-1], 0.0, r[3]) == 0
        d = [oracle.delay(kc, oracle.dm_value(r[0], r[1], r[2] - 1), r[3]) for kc in k[::37]]
        assert all(a <= b for a, b in zip(d, d[1:]))
        d = [oracle.delay(k[-1], oracle.dm_value(r[0], r[1], i), r[3]) for i in range(0, r[2], 13)]
        assert all(a <= b for a, b in zip(d, d[1:]))


def test_pulse_signal_model_equals_search_delay():
    """datagen's pulse sweep (signal model) lands on the oracle's delay for bin 1, so an injected pulse is aligned."""
    for wl in ("tiny", "mid", "ska"):
        w = datagen.get_workload(wl)
        k = oracle.delay_constants(w.freqs_mhz, w.tsamp_s)
        for dm in (0.0, 50.0, 123.456):
            sw = datagen.pulse_sweep(w.freqs_mhz, dm, w.tsamp_s)
            mine = np.array([oracle.delay(kc, dm, 1) for kc in k])
            assert np.max(np.abs(sw - mine)) <= 1 and np.mean(sw == mine) > 0.999


# ------------------------------------------------------------------------------------------------ C3 geometry
def test_chunk_geometry_golden():
    for wl, B, S, n_out, outputs in _rows("geometry.txt"):
        w = datagen.get_workload(wl)
        k = oracle.delay_constants(w.freqs_mhz, w.tsamp_s)
        g = oracle.chunk_geometry(k, w.ranges, w.nsamp)
        assert (g["B"], g["S"], g["n_out"]) == (int(B), int(S), int(n_out))
        assert sum(r[2] * (g["n_out"] // r[3]) for r in w.ranges) == int(outputs)
        assert len(g["chunks"]) == 1


def test_chunk_geometry_streaming_tiles_without_gap():
    w = datagen.get_workload("stream")
    k = oracle.delay_constants(w.freqs_mhz, w.tsamp_s)
    g = oracle.chunk_geometry(k, w.ranges, w.nsamp, chunk_len=1 << 20)
    assert g["S"] == 32384 and g["n_out"] == (1 << 20) - 32384
    pos = 0
    for (start, L, n) in g["chunks"]:
        assert start == pos and L % g["B"] == 0 and start % g["B"] == 0 and start + L <= w.nsamp
        pos += n
    assert len(g["chunks"]) == 10 and g["chunks"][-1][1] == 229272      # SURVEY §8(d) Streaming row
    assert pos == 9342616                                                # SURVEY §8(d) n_out (stream total)


# ------------------------------------------------------------------------------------------------ C4 binning
@pytest.mark.parametrize("b", [1, 2, 4, 8])
def test_binning_constant_and_sum_conservation(b):
    x = np.full((3, 64), 7, np.uint8)
    assert np.all(oracle.bin_time(x, 0, 64 // b, b) == 7 * b)
    rng = np.random.default_rng(b)
    x = rng.integers(0, 256, (5, 96), dtype=np.uint8)
    xb = oracle.bin_time(x, 8, 80 // b, b)
    assert np.array_equal(xb.sum(axis=1), x[:, 8:88].astype(np.int64).sum(axis=1))
    assert np.array_equal(xb, x[:, 8:88].reshape(5, -1, b).astype(np.int64).sum(axis=2))   # numpy reshape-sum
    assert np.all(oracle.bin_time(np.full((1, 16), 255, np.uint8), 0, 2, 8) == 2040)


# ------------------------------------------------------------------------------------------------ C5 dedispersion
def test_dm0_row_is_channel_sum(tiny):
    w, x, k, g = tiny
    xb = oracle.bin_time(x, 0, g["L"], 1)
    D = oracle.dedisperse(xb, k, w.ranges[0], 0, 1, g["n_out"])
    assert np.array_equal(D[0], x[:, :g["n_out"]].astype(np.int64).sum(axis=0))


def test_dedisperse_vs_pure_python_brute_force():
    rng = np.random.default_rng(5)
    C, L = 4, 40
    x = rng.integers(0, 256, (C, L), dtype=np.uint8)
    freqs = np.array([400.0, 390.0, 380.0, 370.0])
    k = oracle.delay_constants(freqs, 1e-3)
    r = (0.0, 0.7, 6, 1)
    dl = [[oracle.delay(k[c], r[0] + i * r[1], 1) for c in range(C)] for i in range(r[2])]
    T = L - max(max(d) for d in dl)
    assert T > 8 and dl[-1][-1] > 3 and len({tuple(d) for d in dl}) > 3       # a non-trivial case
    D = oracle.dedisperse(oracle.bin_time(x, 0, L, 1), k, r, 0, r[2], T)
    for i in range(r[2]):
        for t in range(T):
            assert D[i, t] == sum(int(x[c, t + dl[i][c]]) for c in range(C))


def test_dedisperse_binned_vs_brute_force():
    rng = np.random.default_rng(6)
    C, L, b = 3, 64, 4
    x = rng.integers(0, 256, (C, L), dtype=np.uint8)
    k = oracle.delay_constants(np.array([300.0, 290.0, 280.0]), 1e-3)
    r = (2.0, 1.5, 4, b)
    dl = [[oracle.delay(k[c], r[0] + i * r[1], b) for c in range(C)] for i in range(r[2])]
    T = L // b - max(max(d) for d in dl)
    assert T >= 4 and dl[-1][-1] >= 2
    D = oracle.dedisperse(oracle.bin_time(x, 0, L // b, b), k, r, 0, r[2], T)
    for i in range(r[2]):
        for t in range(T):
            assert D[i, t] == sum(int(x[c, b * (t + dl[i][c]) + j]) for c in range(C) for j in range(b))


def test_dedisperse_constant_input_closed_form():
    w = datagen.get_workload("tiny")
    k = oracle.delay_constants(w.freqs_mhz, w.tsamp_s)
    for b in (1, 2):
        x = np.full((w.nchans, 512), 9, np.uint8)
        r = (0.0, 1.0, 20, b)
        T = 512 // b - oracle.delay(k[-1], 19.0, b)
        D = oracle.dedisperse(oracle.bin_time(x, 0, 512 // b, b), k, r, 0, 20, T)
        assert np.all(D == w.nchans * b * 9)


def test_dedisperse_single_impulse_response():
    w = datagen.get_workload("tiny")
    k = oracle.delay_constants(w.freqs_mhz, w.tsamp_s)
    x = np.zeros((w.nchans, 600), np.uint8)
    c0, t0 = 40, 300
    x[c0, t0] = 200
    r = (0.0, 1.0, 101, 1)
    T = 600 - 65
    D = oracle.dedisperse(oracle.bin_time(x, 0, 600, 1), k, r, 0, 101, T)
    exp = np.zeros_like(D)
    for i in range(101):
        exp[i, t0 - oracle.delay(k[c0], float(i), 1)] = 200
    assert np.array_equal(D, exp)


def test_dedisperse_all_rows_moment_identity(tiny):
    """SURVEY §8(c) pin (v): sum_t D and sum_t t*D from per-channel prefix sums (an O(C) route per row)."""
    w, x, k, g = tiny
    r, T = w.ranges[0], g["n_out"]
    xb = oracle.bin_time(x, 0, g["L"], 1).astype(np.int64)
    D = oracle.dedisperse(oracle.bin_time(x, 0, g["L"], 1), k, r, 0, r[2], T)
    P = np.concatenate([np.zeros((w.nchans, 1), np.int64), np.cumsum(xb, axis=1)], axis=1)
    Q = np.concatenate([np.zeros((w.nchans, 1), np.int64), np.cumsum(xb * np.arange(xb.shape[1]), axis=1)], axis=1)
    tt = np.arange(T)
    for i in range(r[2]):
        d = np.array([oracle.delay(kc, float(i), 1) for kc in k])
        ch = np.arange(w.nchans)
        m0 = (P[ch, T + d] - P[ch, d]).sum()
        m1 = ((Q[ch, T + d] - Q[ch, d]) - d * (P[ch, T + d] - P[ch, d])).sum()
        assert D[i].sum() == m0 and (D[i] * tt).sum() == m1


# ------------------------------------------------------------------------------------------------ C6 statistics
def test_stats_two_valued_row_exact():
    row = np.array([100] * 500 + [104] * 500)             # mean 102, population sigma 2, nothing beyond 3 sigma
    mu, sg, n, it, lo, hi, deg = oracle.row_stats(row)
    assert (mu, sg, n, deg) == (102.0, 2.0, 1000, False) and (lo, hi) == (96, 108) and it == 1


def test_stats_uniform_closed_form():
    M = 200
    row = np.tile(np.arange(M + 1), 7)
    mu, sg, n, *_ = oracle.row_stats(row)
    assert n == row.size and mu == M / 2
    assert abs(sg - np.sqrt(((M + 1) ** 2 - 1) / 12.0)) < 1e-12 * sg


def test_stats_outlier_rejected_hand_worked():
    # 100 x 10 and one 1000: pass 0 mu=19.80, sigma=98.02 -> keep [-274, 313] drops 1000 -> mu=10, sigma=0
    mu, sg, n, it, lo, hi, deg = oracle.row_stats(np.array([10] * 100 + [1000]))
    assert (mu, sg, n) == (10.0, 0.0, 100) and it == 2 and not deg
    # 3:1 mixture of 0 and 40 with a burst of 5 huge samples
    row = np.array(([0] * 3 + [40]) * 250 + [100000] * 5)
    mu, sg, n, *_ = oracle.row_stats(row)
    assert n == 1000 and mu == 10.0 and abs(sg - np.sqrt(300.0)) < 1e-12


def test_stats_gaussian_fixed_point_closed_form():
    """For Gaussian data the 3-sigma clip converges to r*sigma with r^2 = 1 - 2a*phi(a)/(2Phi(a)-1), a = 3r."""
    from math import erf, exp, pi, sqrt
    r = 1.0
    for _ in range(200):
        a = 3.0 * r
        r = sqrt(1.0 - 2.0 * a * (exp(-a * a / 2) / sqrt(2 * pi)) / erf(a / sqrt(2)))
    assert abs(r - 0.98485) < 2e-5                         # the constant SURVEY §8(c) C6 quotes
    rng = np.random.default_rng(3)
    n = 400_000
    row = np.round(rng.normal(520000.0, 1024.0, n)).astype(np.int64)
    mu, sg, cnt, it, *_ = oracle.row_stats(row)
    assert abs(sg / 1024.0 - r) < 4.0 / sqrt(n) and abs(mu - 520000.0) < 5 * 1024 / sqrt(n)
    assert 2 <= it <= 8


def test_stats_order_and_pivot_invariance():
    rng = np.random.default_rng(4)
    row = np.round(rng.normal(8000.0, 130.0, 5000)).astype(np.int64)
    row[::97] += 4000
    a = oracle.row_stats(row)
    b = oracle.row_stats(rng.permutation(row))
    assert a[2:6] == b[2:6]                                # n, iterations, lo, hi identical
    assert abs(a[0] - b[0]) < 1e-9 and abs(a[1] - b[1]) < 1e-9


def test_stats_constant_row_sigma_zero():
    mu, sg, n, it, lo, hi, deg = oracle.row_stats(np.full(300, 77))
    assert (mu, sg, n) == (77.0, 0.0, 300)
    S, wb = oracle.boxcar_snr(np.full(300, 77), [1, 2], mu, sg)
    assert np.all(np.isneginf(S)) and np.all(wb == 0)


# ------------------------------------------------------------------------------------------------ C7 boxcar / SNR
def test_boxcar_hand_worked():
    row = np.array([5, 5, 5, 9, 9, 5, 5, 5])
    S, wb = oracle.boxcar_snr(row, [1, 2, 4], 5.0, 2.0)
    # t=3: w=1 -> (9-5)/2 = 2; w=2 -> (18-10)/(sqrt2*2) = 2*sqrt2; w=4 -> (28-20)/4 = 2
    assert wb[3] == 2 and abs(S[3] - 2 * np.sqrt(2)) < 1e-15
    assert wb[2] == 4 and S[2] == 2.0                      # w=1: 0, w=2: 4/(2*sqrt2)=1.414, w=4: 8/4=2
    assert wb[4] == 1 and S[4] == 2.0                      # w=2: 4/2.83=1.41, w=4: 4/4=1; tie-free
    assert wb[7] == 1 and S[7] == 0.0 and wb[6] == 1       # only w=1 (and 2 at t=6) valid at the end; ties keep smallest
    assert wb[5] == 1 and S[5] == 0.0


def test_boxcar_direct_vs_numpy_convolve_and_prefix():
    rng = np.random.default_rng(8)
    row = rng.integers(500000, 540000, 700).astype(np.int64)
    widths = [1, 2, 3, 8, 64, 256]
    mu, sg = 520000.25, 11000.5
    S, wb = oracle.boxcar_snr(row, widths, mu, sg)
    best = np.full(row.size, -np.inf); bw = np.zeros(row.size, np.int32)
    for w in widths:
        B = np.convolve(row, np.ones(w, np.int64), mode="valid")                 # library routine
        snr = (B - w * mu) / (np.sqrt(w) * sg)
        upd = snr > best[:B.size]
        best[:B.size][upd] = snr[upd]; bw[:B.size][upd] = w
    assert np.array_equal(wb, bw) and np.allclose(S, best, rtol=1e-12, atol=1e-12)
    S2, wb2 = oracle.boxcar_snr(row, widths, mu, sg, prefix=True)
    assert np.array_equal(S, S2) and np.array_equal(wb, wb2)                    # bit-identical routes


# ------------------------------------------------------------------------------------------------ C8 peaks
def test_peaks_hand_built_maps():
    ninf = -np.inf
    S = np.array([[1, 1, 1, 1, 1, 1, 1, 9],
                  [1, 7, 7, 1, 1, 8, 1, 1],
                  [1, 7, 7, 1, 1, 1, 1, 1],
                  [1, 1, 1, 1, ninf, 6.5, 1, 1],
                  [9, 1, 1, 1, ninf, ninf, 1, 6]], dtype=np.float64)
    rr, tt = oracle.find_peaks(S, 6.0)
    got = sorted(zip(rr.tolist(), tt.tolist()))
    # corner (0,7)=9; plateau of 7s -> its first point (1,1) only; (1,5)=8; (3,5)=6.5 next to -inf; corner (4,0)=9;
    # (4,7)=6 is not > threshold 6 (strict)
    assert got == [(0, 7), (1, 1), (1, 5), (3, 5), (4, 0)]
    rr, tt = oracle.find_peaks(S, 6.0, 1, 4)               # halo rows 0 and 4 are neighbours but not reported
    assert sorted(zip(rr.tolist(), tt.tolist())) == [(1, 1), (1, 5), (3, 5)]
    S[0, 6] = 8.5                                          # a bigger neighbour in the halo row kills (1,5)
    rr, tt = oracle.find_peaks(S, 6.0, 1, 4)
    assert sorted(zip(rr.tolist(), tt.tolist())) == [(1, 1), (3, 5)]


# ------------------------------------------------------------------------------------------------ end to end
def test_tiny_injected_pulse_recovered(tiny):
    """BASELINE.json config 1 + north_star 'must recover an injected dispersed pulse at its DM and time within one
    sample'; SURVEY §8(c) C7 closed form SNR ~ A*sqrt(C*w)/16.0026/0.98485 = 12.18 (+- noise)."""
    w, x, k, g = tiny
    xb = oracle.bin_time(x, 0, g["L"], 1)
    r = oracle.search_rows(xb, k, w.ranges[0], 0, g["n_out"], w.widths, w.threshold, 0, 0, w.ranges[0][2],
                           want=("D", "stats"))
    c = r["cands"]
    top = c[np.argmax(c["snr"])]
    assert abs(int(top["dm_index"]) - 50) <= 1 and abs(int(top["sample"]) - 3000) <= 1 and int(top["width"]) == 4
    assert abs(float(top["snr"]) - 12.0 * np.sqrt(64 * 4) / 16.0026 / 0.98485) < 1.5
    assert r["D"][50, 3000:3004].mean() - r["stats"][50, 0] > 4 * r["stats"][50, 1]     # the pulse is in D at t0
    # noise rows: mu ~ 127*C, sigma ~ 0.98485*16.0026*sqrt(C) (SURVEY §8(c) C6 closed form)
    assert abs(np.median(r["stats"][:, 0]) - 127.0 * 64) < 3.0
    assert abs(np.median(r["stats"][:, 1]) / (0.98485 * 16.0026 * 8.0) - 1.0) < 0.02
    # canonical order (range, dm_index, sample)
    key = list(zip(c["dm_index"].tolist(), c["sample"].tolist()))
    assert key == sorted(key)


def test_band_search_equals_full_search(tiny):
    """Searching a band of rows with halo reproduces the same rows of the full search (used for the big configs)."""
    w, x, k, g = tiny
    xb = oracle.bin_time(x, 0, g["L"], 1)
    full = oracle.search_rows(xb, k, w.ranges[0], 0, g["n_out"], w.widths, w.threshold, 0, 0, 101, want=())
    band = oracle.search_rows(xb, k, w.ranges[0], 0, g["n_out"], w.widths, w.threshold, 0, 47, 54, want=())
    sel = full["cands"][(full["cands"]["dm_index"] >= 47) & (full["cands"]["dm_index"] < 54)]
    assert len(sel) > 0 and np.array_equal(sel, band["cands"])


# ------------------------------------------------------------------------------------------------ reading C3x (boxcar-complete chunks)
def test_boxcar_complete_chunks_equal_the_untruncated_definition(tiny):
    """Reading C3x: with E = W_max - 1 extra samples per row, every boxcar that STARTS inside a chunk's output span is
    complete. Pin (independent route): the S map of a chunk equals, position by position, the SNR of numpy boxcar sums
    taken on a row dedispersed over the WHOLE observation, normalised with the chunk's own mu / sigma; and the geometry
    obeys S_x = ceil_B(max_r b_r (delay_max_r + E)), chunks tiling the output axis without gap."""
    w, x, k, g0 = tiny
    widths = w.widths
    E = max(widths) - 1
    rng = w.ranges[0]
    L = 2048
    g = oracle.chunk_geometry(k, w.ranges, w.nsamp, chunk_len=L, boxcar_extra=E)
    assert g["S"] == g0["S"] + E and g["n_out"] == L - g["S"]                     # tiny: bin 1, so S grows by exactly E
    assert [c[0] for c in g["chunks"]] == [j * g["n_out"] for j in range(len(g["chunks"]))]
    xb_all = oracle.bin_time(x, 0, w.nsamp, 1)
    T_all = w.nsamp - g0["S"]
    rows = (0, 50, 100)
    D_all = {i: oracle.dedisperse(xb_all, k, rng, i, i + 1, T_all)[0] for i in rows}
    for (start, Lj, n_out) in g["chunks"][:3]:
        xb = oracle.bin_time(x, start, Lj, 1)
        for i in rows:
            res = oracle.search_rows(xb, k, rng, 0, n_out, widths, w.threshold, start, i, i + 1, want=("D", "stats", "S", "w"), extra=E)
            assert res["D"].shape == (1, n_out + E)
            assert np.array_equal(res["D"][0], D_all[i][start:start + n_out + E])  # D is chunk-invariant, extra samples included
            mu, sg = res["stats"][0]
            m0, s0, *_ = oracle.row_stats(D_all[i][start:start + n_out])           # statistics: the chunk's own span only
            assert (mu, sg) == (m0, s0)
            best = np.full(n_out, -np.inf)
            bw = np.zeros(n_out, np.int32)
            for wd in widths:                                                      # numpy route, no truncation at the chunk end
                B = np.convolve(D_all[i].astype(np.float64), np.ones(wd), mode="valid")[start:start + n_out]
                snr = (B - wd * mu) / (np.sqrt(wd) * sg)
                upd = snr > best + 1e-9
                best[upd] = snr[upd]
                bw[upd] = wd
            assert np.allclose(res["S"][0], best, rtol=1e-9, atol=1e-9)
            assert np.array_equal(res["w"][0][best > 3.0], bw[best > 3.0])
            # and without the extra samples the last W_max - 1 positions are truncated (the behaviour C3x removes)
            old = oracle.search_rows(xb, k, rng, 0, n_out, widths, w.threshold, start, i, i + 1, want=("S",), extra=0)["S"][0]
            assert np.array_equal(old[: n_out - E], res["S"][0][: n_out - E]) or np.allclose(old[: n_out - E], res["S"][0][: n_out - E])


# ------------------------------------------------------------------------------------------------ delay table (helper of the full-size checks)
@pytest.mark.parametrize("wl", ["tiny", "mid", "ska", "lowf"])
def test_delay_table_equals_delay(wl):
    """orc_delay_table is what the all-rows moment identity and the sampled outputs of the full-size GPU tests are built
    from. Pin: its [i][c] entry is orc_delay(k[c], DM_i, bin) on a scatter of (range, i, c) that includes the corners, and
    an (i, c) transposition or a dropped `bin` cannot pass (the scatter has i != c and binned ranges)."""
    w = datagen.get_workload(wl)
    k = oracle.delay_constants(w.freqs_mhz, w.tsamp_s)
    rs = np.random.default_rng(17)
    for r in w.ranges:
        i0 = int(rs.integers(0, max(1, r[2] - 40)))
        i1 = min(r[2], i0 + 40)
        tab = oracle.delay_table(k, r, i0, i1)
        assert tab.shape == (i1 - i0, w.nchans) and tab.dtype == np.int64
        cs = np.concatenate([[0, 1, w.nchans - 1], rs.integers(0, w.nchans, 50)])
        js = np.concatenate([[i0, i1 - 1, i0], rs.integers(i0, i1, 50)])
        for c, i in zip(cs, js):
            assert tab[int(i) - i0, int(c)] == oracle.delay(k[int(c)], oracle.dm_value(r[0], r[1], int(i)), r[3]), (wl, r, i, c)
        # whole-table form (i0 = 0, i1 = ndms) agrees with the slice form
        if r[2] <= 2500:
            assert np.array_equal(oracle.delay_table(k, r)[i0:i1], tab)


def test_delay_table_reproduces_the_golden_delays():
    """The 25 closed-form rows of tests/golden/delays.txt (SURVEY §8(c) 'C2 delays'), read through the table form: the DM of
    each golden row is located in the workload's DM plan and the entry [i][c] must be the golden value."""
    n = 0
    for wl, c, dm, b, exp in _rows("delays.txt"):
        w = datagen.get_workload(wl)
        k = oracle.delay_constants(w.freqs_mhz, w.tsamp_s)
        for r in w.ranges:
            if r[3] != int(b):
                continue
            i = int(round((float(dm) - r[0]) / r[1]))
            if 0 <= i < r[2] and oracle.dm_value(r[0], r[1], i) == float(dm):
                assert oracle.delay_table(k, r, i, i + 1)[0, int(c)] == int(exp), (wl, c, dm, b)
                n += 1
    assert n >= 15          # most golden rows lie on a DM trial of their workload's plan


# ------------------------------------------------------------------------------------------------ C9 record
def _c9_workload():
    """Tiny's band with a bin-1 and a bin-4 range, 4 chunks of 4096 samples, two bright pulses whose place is fixed by the
    INJECTION (datagen), not by the oracle: pulse A at DM 20 (range 0, bin 1), t0 = 5000, 4 samples wide -> chunk 1;
    pulse B at DM 70 (range 1, bin 4, dm_index 15), t0 = 9000, 16 samples wide -> chunk 2."""
    base = datagen.get_workload("tiny")
    return datagen.scaled(base, name="tiny_c9", nsamp=16384, ranges=((0.0, 1.0, 40, 1), (40.0, 2.0, 30, 4)), widths=(1, 2, 4, 8, 16),
                          fixed_pulses=((20.0, 5000, 4, 14.0), (70.0, 9000, 16, 8.0)))


def test_candidate_record_in_binned_ranges_and_later_chunks():
    """Reading C9: sample = chunk_start + bin*t', width = bin*w*. Pin: pulses injected at known UNBINNED samples, widths and
    DMs in a bin-4 range and in chunks 1 and 2 of a chunked geometry must come back at those unbinned coordinates (a
    dropped `bin` factor would report sample ~ 8064 + 234 and width 4; a dropped chunk_start would report sample < 4096)."""
    w = _c9_workload()
    pl, dms, dl = w.pulses()
    x = datagen.generate(w.seed, w.nchans, w.nsamp, pl, dl)
    k = oracle.delay_constants(w.freqs_mhz, w.tsamp_s)
    g = oracle.chunk_geometry(k, w.ranges, w.nsamp, chunk_len=4096)
    assert g["B"] == 4 and g["S"] % 4 == 0 and len(g["chunks"]) >= 4
    found = {}
    for (r_index, t0, width, dm_index) in ((0, 5000, 4, 20), (1, 9000, 16, 15)):
        rng = w.ranges[r_index]
        b = rng[3]
        j = t0 // g["n_out"]
        start, Lj, n_out = g["chunks"][j]
        assert start == j * g["n_out"] and start <= t0 < start + n_out and j >= 1
        xb = oracle.bin_time(x, start, Lj // b, b)
        res = oracle.search_rows(xb, k, rng, r_index, n_out // b, w.widths, w.threshold, start, 0, rng[2], want=())
        c = res["cands"]
        assert len(c) > 0
        top = c[np.argmax(c["snr"])]
        found[r_index] = top
        assert int(top["range"]) == r_index and abs(int(top["dm_index"]) - dm_index) <= 1
        assert abs(int(top["sample"]) - t0) <= b, (int(top["sample"]), t0)                  # unbinned, absolute
        assert int(top["sample"]) >= start and (int(top["sample"]) - start) % b == 0
        assert int(top["width"]) % b == 0 and width // 2 <= int(top["width"]) <= 2 * width, int(top["width"])
        assert float(top["dm"]) == np.float32(oracle.dm_value(rng[0], rng[1], int(top["dm_index"])))
        assert np.all(c["sample"] >= start) and np.all(c["sample"] < start + n_out)          # every record is inside its chunk
    assert float(found[0]["snr"]) > 10 and float(found[1]["snr"]) > 10


def test_threshold_is_compared_as_a_float32_value():
    """The C ABI takes the threshold as float (include/aa.h) and widens it; the tests hand the oracle np.float32(threshold)
    so both sides compare against the same double. 6.1 is not float-exact: the two doubles differ, and a row built to sit
    between them shows which one is in force."""
    t32, t64 = float(np.float32(6.1)), 6.1
    assert t32 != t64 and t32 < t64
    S = np.full((1, 5), -np.inf)
    S[0, 2] = (t32 + t64) / 2                       # above float32(6.1), below the double 6.1
    assert len(oracle.find_peaks(S, t32)[0]) == 1 and len(oracle.find_peaks(S, t64)[0]) == 0


# ------------------------------------------------------------------------------------------------ the parallel harness of the full-size check
def test_sliced_parallel_oracle_equals_the_single_call(tiny):
    """tests/helpers.run_oracle_slices (DM slices in a process pool, the route of the SKA-like full-oracle GPU test) returns,
    slice by slice, exactly what ONE oracle.search_rows call over the whole range returns: statistics, D (through the
    row hashes) and candidates. Pins the slicing, the halo handling and the gathering, not the oracle."""
    from helpers import oracle_slices, row_hash, run_oracle_slices
    w, x, k, g = tiny
    chunk = g["chunks"][0]
    full = oracle.search_rows(oracle.bin_time(x, 0, g["L"], 1), k, w.ranges[0], 0, g["n_out"], w.widths,
                              float(np.float32(w.threshold)), 0, 0, w.ranges[0][2], want=("D", "stats"))
    slices = oracle_slices(w.ranges, rows_per_unit_cost=16)
    assert [s[1] for s in slices] == list(range(0, 101, 16)) and slices[-1][2] == 101
    res = run_oracle_slices(w, x, chunk, slices, processes=2)
    cands = []
    for (r, i0, i1) in slices:
        st, hs, c = res[(r, i0, i1)]
        assert np.array_equal(st, full["stats"][i0:i1])
        assert hs == [row_hash(full["D"][i]) for i in range(i0, i1)]
        cands.append(c)
    assert np.array_equal(np.concatenate(cands), full["cands"])
    assert row_hash(full["D"][3]) != row_hash(full["D"][4])


# ------------------------------------------------------------------------------------------------ reading C7m (per-width measured statistics)
def test_per_width_stats_width_one_is_reading_c7_bit_for_bit():
    rng = np.random.default_rng(21)
    row = np.round(rng.normal(52000.0, 410.0, 6000)).astype(np.int64)
    row[1000:1004] += 3000
    mu, sg, *_ = oracle.row_stats(row)
    S1, w1 = oracle.boxcar_snr(row, [1], mu, sg)
    Sm, wm, ws = oracle.boxcar_snr_perwidth(row, len(row), [1])
    assert np.array_equal(S1, Sm) and np.array_equal(w1, wm) and (ws[0, 0], ws[0, 1], ws[0, 2]) == (mu, sg, float(row[0]))
    # in a longer width list the width-1 statistics are unchanged and each width's p_w is its first boxcar sum
    _, _, ws = oracle.boxcar_snr_perwidth(row, len(row), [1, 2, 5, 32])
    assert (ws[0, 0], ws[0, 1]) == (mu, sg)
    assert [ws[i, 2] for i in range(4)] == [float(row[:w].sum()) for w in (1, 2, 5, 32)]


def test_per_width_stats_hand_worked():
    # w = 2 sums are constant -> sigma_2 = 0 -> width 2 is skipped; width 1: mean 2, sigma 1
    S, wb, ws = oracle.boxcar_snr_perwidth(np.array([1, 3] * 4), 8, [1, 2])
    assert ws[1, 1] == 0.0 and np.all(wb == 1) and np.array_equal(S, np.array([-1.0, 1.0] * 4))
    # row 0 0 4 0 0 0 4 0 0: B_2 = 0 4 4 0 0 4 4 0 -> mean 2, sigma 2 exactly; B_1: mean 8/9, var 224/81
    row = np.array([0, 0, 4, 0, 0, 0, 4, 0, 0])
    S, wb, ws = oracle.boxcar_snr_perwidth(row, 9, [1, 2])
    assert (ws[1, 0], ws[1, 1], ws[1, 2]) == (2.0, 2.0, 0.0)
    assert abs(ws[0, 0] - 8 / 9) < 1e-15 and abs(ws[0, 1] - np.sqrt(224.0) / 9) < 1e-15
    s1 = (4 - 8 / 9) / (np.sqrt(224.0) / 9)                # 1.871 > 1: width 1 wins on the spikes
    s0 = (0 - 8 / 9) / (np.sqrt(224.0) / 9)                # -0.534: beats SNR_2 = -1 where B_2 = 0, loses to SNR_2 = +1 where B_2 = 4
    assert wb.tolist() == [1, 2, 1, 1, 1, 2, 1, 1, 1]      # SNR_2 = -1 1 1 -1 -1 1 1 -1; the last position has only w = 1
    assert abs(S[2] - s1) < 1e-14 and S[1] == 1.0 and S[5] == 1.0 and abs(S[0] - s0) < 1e-14 and abs(S[8] - s0) < 1e-14
    # with E extra samples present (reading C3x) every start position t < T has a complete boxcar: n_w = T
    S2, wb2, ws2 = oracle.boxcar_snr_perwidth(np.array([0, 0, 4, 0, 0, 0, 4, 0, 0, 0]), 9, [1, 2])
    assert len(S2) == 9 and abs(ws2[1, 0] - 16 / 9) < 1e-15            # B_2 = 0 4 4 0 0 4 4 0 0: nine sums, mean 16/9
    assert (ws2[0, 0], ws2[0, 1]) == (ws[0, 0], ws[0, 1])              # width-1 statistics still use the first T samples only


def test_per_width_stats_white_noise_closed_form():
    """White Gaussian rows: sigma_w -> 0.98485 * sigma * sqrt(w), mu_w -> w * mu (SURVEY §8(c) C6 fixed point applied to B_w),
    i.e. C7m reduces to C7 where C7's assumption holds; the estimate's scatter grows with w (n/w independent sums)."""
    rng = np.random.default_rng(22)
    n, sig = 400_000, 700.0
    row = np.round(rng.normal(3.0e6, sig, n)).astype(np.int64)
    widths = [1, 2, 4, 16, 64]
    S, wb, ws = oracle.boxcar_snr_perwidth(row, n, widths)
    for iw, w in enumerate(widths):
        assert abs(ws[iw, 1] / (0.98485 * sig * np.sqrt(w)) - 1.0) < 5.0 * np.sqrt(w / (2.0 * n)) + 2e-3, (w, ws[iw])
        assert abs(ws[iw, 0] - w * 3.0e6) < 6.0 * sig * w / np.sqrt(n)


def test_per_width_stats_red_noise_where_sqrt_w_scaling_is_wrong():
    """AR(1) noise x_t = rho x_(t-1) + e_t: Var(sum of w samples) = s^2 [w + 2 sum_{k=1}^{w-1} (w-k) rho^k] (textbook
    autocovariance s^2 rho^k). The measured sigma_w follows it; the sqrt(w) scaling of the width-1 sigma (reading C7) is
    low by more than a factor 2 at w = 16, rho = 0.9 - the case C7m exists for."""
    rng = np.random.default_rng(23)
    n, rho, s_e = 600_000, 0.9, 200.0
    e = rng.normal(0.0, s_e, n)
    x = np.empty(n)
    acc = 0.0
    for t in range(n):
        acc = rho * acc + e[t]
        x[t] = acc
    row = np.round(x + 1.0e6).astype(np.int64)
    s_x = s_e / np.sqrt(1 - rho * rho)
    widths = [1, 4, 16]
    _, _, ws = oracle.boxcar_snr_perwidth(row, n, widths)
    for iw, w in enumerate(widths):
        var_w = s_x ** 2 * (w + 2.0 * sum((w - k) * rho ** k for k in range(1, w)))
        assert abs(ws[iw, 1] / (0.98485 * np.sqrt(var_w)) - 1.0) < 0.04, (w, ws[iw, 1], np.sqrt(var_w))
    assert ws[2, 1] > 2.0 * np.sqrt(16.0) * ws[0, 1]          # sqrt(w) scaling underestimates sigma_16 by > 2x


def test_per_width_stats_invariant_under_a_constant_shift():
    """All arithmetic is about the pivots p_w, so adding a constant to D changes the SNR only through the rounding of
    mu_w = p_w + S1/n (about 1e-10 relative here) and never the chosen width or the integer statistics."""
    rng = np.random.default_rng(24)
    row = np.round(rng.normal(0.0, 90.0, 5000)).astype(np.int64)
    row[2000:2010] += 700
    a = oracle.boxcar_snr_perwidth(row + 4096, len(row), [1, 2, 8, 32])
    b = oracle.boxcar_snr_perwidth(row + 8_000_000, len(row), [1, 2, 8, 32])
    assert np.allclose(a[0], b[0], rtol=1e-8, atol=1e-8) and np.array_equal(a[1], b[1]) and np.array_equal(a[2][:, 1], b[2][:, 1])
    assert np.array_equal(a[2][:, 2] - np.array([1, 2, 8, 32]) * 4096.0, b[2][:, 2] - np.array([1, 2, 8, 32]) * 8.0e6)   # p_w shifts by w * c
    assert a[1][2000] in (8, 32) and a[0][2000] > 10


def test_per_width_stats_end_to_end_recovers_the_injected_pulse(tiny):
    w, x, k, g = tiny
    xb = oracle.bin_time(x, 0, g["L"], 1)
    a = oracle.search_rows(xb, k, w.ranges[0], 0, g["n_out"], w.widths, w.threshold, 0, 0, 101, want=())["cands"]
    b = oracle.search_rows(xb, k, w.ranges[0], 0, g["n_out"], w.widths, w.threshold, 0, 0, 101, want=(), per_width=True)["cands"]
    ta, tb = a[np.argmax(a["snr"])], b[np.argmax(b["snr"])]
    assert (int(tb["dm_index"]), int(tb["sample"]), int(tb["width"])) == (int(ta["dm_index"]), int(ta["sample"]), int(ta["width"]))
    assert abs(float(tb["snr"]) / float(ta["snr"]) - 1.0) < 0.05          # white noise: the two readings nearly agree


# ------------------------------------------------------------------------------------------------ 16-bit input samples
def test_bin16_constant_conservation_and_numpy_reshape_sum():
    """orc_bin16 (uint16 input): constant input v gives b*v; the sum over t' equals the sum over t; and every binned value
    equals numpy's reshape-sum of the same samples, for every b, on values that need all 12 bits and a strided view."""
    rs = np.random.default_rng(16)
    big = rs.integers(0, 4096, size=(7, 1000), dtype=np.uint16)
    x = big[:, 3:963]                                                   # rows are not contiguous with each other
    for b in (1, 2, 4, 8):
        nb = 900 // b
        got = oracle.bin_time(x, 40, nb, b)
        exp = x[:, 40:40 + nb * b].astype(np.int64).reshape(7, nb, b).sum(axis=2)
        assert got.dtype == np.uint16 and np.array_equal(got.astype(np.int64), exp)
        assert int(got.astype(np.int64).sum()) == int(x[:, 40:40 + nb * b].astype(np.int64).sum())
        const = np.full((3, 64), 4095, np.uint16)
        assert np.all(oracle.bin_time(const, 0, 64 // b, b) == 4095 * b)
    with pytest.raises(AssertionError):                                  # 8 * 9000 does not fit the uint16 a sum is held in
        oracle.bin_time(np.full((2, 64), 9000, np.uint16), 0, 8, 8)


def test_dedispersion_of_16bit_input_brute_force_and_dm0_channel_sum():
    """The whole chain on a 16-bit array: D of every row equals a pure-Python triple loop written from the north_star
    formula (bin 1 and bin 2), and the DM = 0 row is the channel sum."""
    rs = np.random.default_rng(1616)
    C, N = 6, 400
    x = rs.integers(0, 4096, size=(C, N), dtype=np.uint16)
    freqs = 1400.0 - 25.0 * np.arange(C)
    tsamp = 1e-3
    k = oracle.delay_constants(freqs, tsamp)
    for b, rng in ((1, (0.0, 3.0, 9, 1)), (2, (5.0, 4.0, 6, 2))):
        nb = N // b
        xb = oracle.bin_time(x, 0, nb, b)
        dmax = oracle.delay(k[-1], oracle.dm_value(rng[0], rng[1], rng[2] - 1), b)
        T = nb - dmax
        D = oracle.dedisperse(xb, k, rng, 0, rng[2], T)
        for i in range(rng[2]):
            dm = rng[0] + i * rng[1]
            for t in range(0, T, 7):
                acc = 0
                for c in range(C):
                    d = int(np.floor(4.148808e3 * dm * (freqs[c] ** -2 - freqs[0] ** -2) / tsamp / b + 0.5))
                    for j in range(b):
                        acc += int(x[c, b * (t + d) + j])
                assert int(D[i, t]) == acc, (b, i, t)
    xb = oracle.bin_time(x, 0, N, 1)
    D0 = oracle.dedisperse(xb, k, (0.0, 1.0, 1, 1), 0, 1, N)
    assert np.array_equal(D0[0], x.astype(np.int64).sum(axis=0))


def test_generator_16bit_matches_its_recipe():
    """datagen 16-bit mode: same Gaussian draws as the 8-bit recipe (same seed => (x16 - mean16) == (x8 - mean8) wherever
    neither clips), clipped to the stated bit depth."""
    a = datagen.generate(77, 5, 4096, mean=127.0, sigma=16.0)
    b = datagen.generate(77, 5, 4096, mean=1800.0, sigma=16.0, bits=16, max_value=4095)
    assert b.dtype == np.uint16 and int(b.max()) <= 4095
    ok = (a > 0) & (a < 255)
    assert np.array_equal(a[ok].astype(np.int64) - 127, b[ok].astype(np.int64) - 1800)
    c = datagen.generate(77, 5, 4096, mean=4090.0, sigma=16.0, bits=16, max_value=4095)
    assert int(c.max()) == 4095 and np.mean(c == 4095) > 0.3


def test_moment_helpers_equal_the_moments_of_the_oracle_rows():
    """tests/helpers.py derives sum_t D and sum_t t*D of every row from prefix sums of the INPUT (the all-rows check of the
    full-size GPU tests). Here both helpers are held against the moments of the rows the oracle dedisperses, on a case with
    three binning factors, a chunk that starts inside the observation and channel blocks that do not divide the channel count."""
    from helpers import row_moments_all_ranges, row_moments_from_input
    rs = np.random.default_rng(77)
    C, N = 37, 4096
    x = rs.integers(0, 256, size=(C, N), dtype=np.uint8)
    freqs = 1400.0 - 0.7 * np.arange(C)
    k = oracle.delay_constants(freqs, 512e-6)
    ranges = ((0.0, 0.8, 9, 1), (7.2, 1.6, 5, 2), (15.2, 3.0, 4, 4))
    start, length, n_out = 256, 3200, 2400
    allr = row_moments_all_ranges(x, k, ranges, start, length, n_out, chan_block=8, threads=2)
    for r, rng in enumerate(ranges):
        b, T = rng[3], n_out // rng[3]
        xb = oracle.bin_time(x, start, length // b, b)
        D = oracle.dedisperse(xb, k, rng, 0, rng[2], T).astype(np.int64)
        m0, m1 = D.sum(axis=1), (D * np.arange(T, dtype=np.int64)).sum(axis=1)
        assert np.array_equal(allr[r][0], m0) and np.array_equal(allr[r][1], m1), r
        e0, e1 = row_moments_from_input(x, k, rng, start, length, T)
        assert np.array_equal(e0, m0) and np.array_equal(e1, m1), r
