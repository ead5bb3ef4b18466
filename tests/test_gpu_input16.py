"""GPU parity for 16-bit input samples (SURVEY §8(f1); PAPER.md:47 step 1, :67): the same definitions on uint16 filterbanks.
The oracle side is orc_bin16 -> the unchanged dedispersion / SPS chain; the CUDA side turns the chunk into per-channel offset
forms (k_input16.cu) that ride the 1-byte (bin 1, 2, 4) and uint16 (bin 8) paths of K2, with exactly scattered exceptions and a
global-memory kernel for exception-heavy chunks. Bars as everywhere: D bit-exact, mu/sigma ==, candidate lists identical."""
import numpy as np
import pytest

import datagen
from datagen.workloads import Workload, scaled

from helpers import GpuRun, OracleRun, check_band, compare_candidates, make_input

pytestmark = pytest.mark.gpu


def _every_row(w, x, **kw):
    gpu, orc = GpuRun(w, x, **kw), OracleRun(w, x)
    try:
        exp_all = []
        for j, chunk in enumerate(gpu.chunks):
            gpu.dedisperse()
            status = gpu.sps()
            assert status == (gpu.aa.AA_STATUS_FINISHED if j == len(gpu.chunks) - 1 else gpu.aa.AA_STATUS_CHUNK_DONE)
            for r, rng in enumerate(w.ranges):
                exp_all.append(check_band(gpu, orc, chunk, r, 0, rng[2], after_sps=True))
        got = gpu.candidates(allow_overflow=True)
        exp = np.concatenate(exp_all)
        n, og, oe = compare_candidates(got, exp, w.threshold)
        assert n + og == len(got) and n + oe == len(exp)
        return gpu.info, got, gpu.aa.aa_strategy_describe(gpu.h)
    finally:
        gpu.close()


@pytest.mark.parametrize("nchans,nsamp,ranges,kw", [
    (61, 5003, ((0.0, 1.3, 37, 1), (48.1, 2.6, 5, 2), (61.1, 5.0, 33, 4), (226.1, 9.0, 3, 8)), {}),       # nothing a multiple of a tile
    (61, 20011, ((0.0, 1.3, 37, 1), (48.1, 2.6, 5, 2), (61.1, 5.0, 33, 4), (226.1, 9.0, 3, 8)), {"chunk_len_hint": 6000}),   # chunks + prefetch
    (1, 2100, ((0.0, 1.0, 3, 1),), {}),                                                                      # one channel: D == x
    (300, 9000, ((0.0, 0.5, 65, 2), (32.5, 1.0, 31, 8)), {}),                                                # > 256 channels: 16-bit carries
    (300, 30000, ((0.0, 0.5, 65, 2), (10.0, 0.5, 40, 1)), {"time_major": True, "chunk_len_hint": 8000}),     # corner turn of uint16 samples
    (67, 5003, ((0.0, 1.3, 37, 1), (226.1, 9.0, 3, 8)), {"time_major": True}),                               # odd channel count, time-major
])
def test_16bit_ragged_shapes_every_row(nchans, nsamp, ranges, kw):
    """12-bit-deep samples N(1800, 16) + pulses in uint16: every row, statistic and candidate equals the oracle's."""
    w = Workload("ragged16", nchans, 420.0, -100.0 / max(nchans, 2), 2048e-6, nsamp, ranges, (1, 2, 3, 7, 16), 5.0,
                 seed=177 + nchans, npulses=3, pulse_dm=(5.0, 60.0), pulse_width_max=8, pulse_snr=(10.0, 25.0),
                 noise_mean=1800.0, input_bits=16, max_value=4095)
    x, _ = make_input(w)
    assert x.dtype == np.uint16 and int(x.max()) > 1500
    before = datagen.checksum(x)
    info, got, desc = _every_row(w, x, **kw)
    assert datagen.checksum(x) == before and info["input_bits"] == 16 and info["input_max"] == 4095 and len(got) > 0
    assert "offset-uint8 route" in desc


@pytest.mark.parametrize("kind", ["uniform_dense", "mixed_groups", "wide_noise"])
def test_16bit_exception_heavy_chunks_take_the_global_memory_route_bit_exact(kind):
    """Uniform 12-bit samples (nearly every sample an exception), channel groups that choose different routes within one chunk,
    and noise too wide for the byte window (sigma 60: bin 1 stays sparse, the binned forms do not): every row equals the oracle."""
    rs = np.random.default_rng(1604)
    C, N = (320, 12_000) if kind == "mixed_groups" else (24, 30_000)
    gauss = np.clip(np.floor(2000.0 + 16.0 * rs.standard_normal((C, N)) + 0.5), 0, 4095).astype(np.uint16)
    unif = rs.integers(0, 4096, size=(C, N), dtype=np.uint16)
    if kind == "uniform_dense":
        x = unif
    elif kind == "mixed_groups":
        x = np.where((np.arange(C) < 256)[:, None], gauss, unif).astype(np.uint16)
    else:
        x = np.clip(np.floor(2000.0 + 60.0 * rs.standard_normal((C, N)) + 0.5), 0, 4095).astype(np.uint16)
    nd = 600
    w = Workload(kind, C, 1500.0, -0.5, 256e-6, N, ((0.0, 0.01, nd, 1), (6.0, 0.01, nd, 2), (30.0, 0.02, nd, 8)), (1, 2, 4), 6.0, seed=1,
                 npulses=0, pulse_dm=(0.0, 0.0), pulse_width_max=1, input_bits=16, max_value=4095)
    gpu, orc = GpuRun(w, x), OracleRun(w, x)
    try:
        gpu.dedisperse()
        for r, rng in enumerate(w.ranges):
            for (i0, i1) in ((0, 3), (nd // 2, nd // 2 + 3), (nd - 3, nd)):
                check_band(gpu, orc, gpu.chunks[0], r, i0, i1, after_sps=False)
        gpu.sps()
    finally:
        gpu.close()


def test_16bit_extreme_values_are_exact():
    """All-max and all-zero 16-bit inputs (closed form D = C*b*v) and the largest value a bin-8 plan admits (8191)."""
    for v, mx in ((4095, 4095), (0, 4095), (8191, 8191)):
        w = Workload("const16", 1024, 1500.0, -0.25, 64e-6, 6000, ((0.0, 2.0, 40, 1), (80.0, 4.0, 33, 8)), (1, 4), 6.0,
                     seed=1, npulses=0, pulse_dm=(0.0, 0.0), pulse_width_max=1, input_bits=16, max_value=mx)
        x = np.full((w.nchans, w.nsamp), v, np.uint16)
        gpu = GpuRun(w, x)
        try:
            gpu.dedisperse()
            for r, rng in enumerate(w.ranges):
                for i in (0, rng[2] // 2, rng[2] - 1):
                    assert np.all(gpu.row(r, i).astype(np.int64) == w.nchans * rng[3] * v)
            gpu.sps()
            assert len(gpu.candidates()) == 0
        finally:
            gpu.close()


def test_16bit_boxcar_sums_beyond_int32_are_an_error_not_a_wrong_candidate():
    """A 16-bit plan has no plan-time bound on boxcar sums (include/aa.h, aa_plan_set_input_bits): square-wave data whose widest
    boxcar times the largest |D - D[0]| reaches 2^31 must end in AA_ERR_RANGE (sticky), and D itself is still exact."""
    import paper_1912_07704_b200 as aa
    C, N = 128, 8192
    x = np.zeros((C, N), np.uint16)
    x[:, 2048:6144] = 65535                                       # |D - D[0]| = 128 * 65535 = 8.4e6; x 512 = 4.3e9 > 2^31
    w = Workload("square16", C, 1500.0, -0.5, 256e-6, N, ((0.0, 1.0, 20, 1),), (1, 8, 64, 512), 6.0, seed=1, npulses=0, pulse_dm=(0.0, 0.0),
                 pulse_width_max=1, input_bits=16, max_value=65535)
    gpu, orc = GpuRun(w, x), OracleRun(w, x)
    try:
        gpu.dedisperse()
        check_band(gpu, orc, gpu.chunks[0], 0, 0, 20, after_sps=False)
        gpu.sps()
        with pytest.raises(aa.AaError) as e:
            gpu.candidates()
        assert e.value.status == aa.AA_ERR_RANGE and "2^31" in e.value.message
        with pytest.raises(aa.AaError) as e:                        # sticky
            gpu.dedisperse()
        assert e.value.status == aa.AA_ERR_RANGE
    finally:
        gpu.close()
    # the same data with a narrow width list is fine: 8 * 8.4e6 < 2^31
    w2 = scaled(w, widths=(1, 8), name="square16_narrow")
    info, got, _ = _every_row(w2, x)
    assert info["input_bits"] == 16


def test_16bit_sample_above_max_value_is_an_error_not_a_wrong_row():
    """The plan states max_value = 4095; ONE sample of the chunk is 4096. K1 packs binned sums into 16-bit lanes that rely on the
    bound, so the chunk must end in AA_ERR_RANGE (sticky) naming max_value, on the offset-form route and on the route of an
    exception-heavy chunk alike; the same data under a plan that admits the value runs clean."""
    import paper_1912_07704_b200 as aa
    for sigma in (16.0, 600.0):                                    # 600: every group is over the exception rate (global-memory route)
        w = Workload("range16", 256, 1500.0, -0.5, 64e-6, 20000, ((0.0, 1.0, 24, 1), (24.0, 2.0, 16, 4)), (1, 4), 6.0, seed=5, npulses=0,
                     pulse_dm=(0.0, 0.0), pulse_width_max=1, noise_mean=1800.0, noise_sigma=sigma, input_bits=16, max_value=4095)
        x, _ = make_input(w)
        assert int(x.max()) <= 4095
        x[131, 7777] = 4096
        gpu = GpuRun(w, x)
        try:
            gpu.dedisperse()
            gpu.sps()
            with pytest.raises(aa.AaError) as e:
                gpu.candidates()
            assert e.value.status == aa.AA_ERR_RANGE and "max_value = 4095" in e.value.message
            with pytest.raises(aa.AaError) as e:                    # sticky
                gpu.dedisperse()
            assert e.value.status == aa.AA_ERR_RANGE
        finally:
            gpu.close()
        info, got, _ = _every_row(scaled(w, max_value=8191, name="range16_wider"), x)
        assert info["input_max"] == 8191


def test_16bit_device_entry_point_and_host_array_checks():
    """aa_run_dedispersion_device with a resident uint16 chunk gives the host-path result; the binding refuses a uint8 array for
    a 16-bit plan (and vice versa) instead of reading it as raw bytes."""
    import torch
    w = Workload("dev16", 64, 1500.0, -1.0, 256e-6, 8192, ((0.0, 1.0, 50, 1), (50.0, 2.0, 20, 4)), (1, 2, 4, 8), 6.0, seed=5, npulses=2,
                 pulse_dm=(5.0, 60.0), pulse_width_max=8, pulse_snr=(10.0, 20.0), noise_mean=900.0, input_bits=16, max_value=4095)
    x, _ = make_input(w)
    gpu = GpuRun(w, x)
    try:
        ref = gpu.st.run(x)
        gpu.aa.aa_strategy_reset(gpu.h)
        xd = torch.from_numpy(x.view(np.int16)).cuda()
        gpu.aa.aa_run_dedispersion_device(gpu.h, xd)
        gpu.sps()
        got = gpu.candidates()
        assert len(got) == len(ref) > 0 and all(np.array_equal(got[f], ref[f]) for f in ref.dtype.names)
        gpu.aa.aa_strategy_reset(gpu.h)
        with pytest.raises(TypeError):
            gpu.aa.aa_run_dedispersion(gpu.h, x.astype(np.uint8))
    finally:
        gpu.close()
    w8 = datagen.get_workload("tiny")
    x8, _ = make_input(w8)
    g8 = GpuRun(w8, x8)
    try:
        with pytest.raises(TypeError):
            g8.aa.aa_run_dedispersion(g8.h, x8.astype(np.uint16))
        with pytest.raises(ValueError):
            g8.aa.aa_run_dedispersion(g8.h, np.ascontiguousarray(x8.T))
    finally:
        g8.close()
