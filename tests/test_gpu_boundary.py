"""GPU tests of the boundary behaviour the paper asks of the API and of the rarely taken routes of the kernels:
memory manager (one allocation, no leak, caller-lent arena: PAPER.md:33), ownership of results, immutable
strategy, status codes per iteration, candidate overflow, and the fallback route of K3
(rows whose head is not representative of the row) — all compared with the oracle where there is arithmetic."""
import numpy as np
import pytest

import datagen
from datagen.workloads import Workload, scaled

from helpers import GpuRun, OracleRun, check_band, compare_candidates, make_input

pytestmark = pytest.mark.gpu


def _free_bytes():
    import torch
    torch.cuda.synchronize()
    return torch.cuda.mem_get_info()[0]


def test_one_allocation_no_leak_and_lent_arena():
    import torch
    import paper_1912_07704_b200 as aa
    torch.cuda.init()
    torch.zeros(1, device="cuda")
    w = datagen.get_workload("tiny")
    x, _ = make_input(w)
    warm = GpuRun(w, x)                 # first use loads the kernels and creates the context's pools: not part of the check
    warm.st.run(x)
    warm.close()
    before = _free_bytes()
    g = GpuRun(w, x)
    try:
        info = g.info
        assert info["owns_arena"] == 1 and info["arena_bytes_total"] == info["arena_bytes_used"] > 0
        during = _free_bytes()
        assert before - during >= info["arena_bytes_used"]                 # the single cudaMalloc (+ allocator granularity)
        ref = g.st.run(x)
        assert _free_bytes() == during                                     # nothing is allocated by aa_run_*
    finally:
        g.close()
    assert _free_bytes() == before                                         # proper de-allocation
    # caller-lent arena: a torch tensor; the library allocates nothing on the device
    need = info["arena_bytes_used"]
    arena = torch.empty(need + 4096, dtype=torch.uint8, device="cuda")
    base = _free_bytes()
    g2 = GpuRun(w, x, arena=arena)
    try:
        assert g2.info["owns_arena"] == 0 and _free_bytes() == base
        got = g2.st.run(x)
        assert _free_bytes() == base
        assert len(got) == len(ref) and all(np.array_equal(got[f], ref[f]) for f in ref.dtype.names)
    finally:
        g2.close()
    small = torch.empty(need // 2, dtype=torch.uint8, device="cuda")
    with pytest.raises(aa.AaError) as e:
        GpuRun(w, x, arena=small)
    assert e.value.status == aa.AA_ERR_BUDGET_TOO_SMALL and "needs" in e.value.message     # states the bytes required


def test_status_codes_order_and_immutable_strategy():
    import paper_1912_07704_b200 as aa
    w = scaled(datagen.get_workload("tiny"), nsamp=6000, name="tiny6k")
    x, _ = make_input(w)
    g = GpuRun(w, x, chunk_len_hint=2048)
    try:
        n = g.info["nchunks"]
        assert n >= 3
        desc0 = aa.aa_strategy_describe(g.h)
        geo0 = [aa.aa_strategy_get_range_info(g.h, r) for r in range(len(w.ranges))]
        with pytest.raises(aa.AaError) as e:                               # "another module still needs to run"
            aa.aa_run_sps(g.h)
        assert e.value.status == aa.AA_ERR_ORDER
        seen = []
        for j in range(n):
            assert aa.aa_run_dedispersion(g.h, x) == aa.AA_OK
            with pytest.raises(aa.AaError) as e:
                aa.aa_run_dedispersion(g.h, x)                             # SPS of this chunk has not run yet
            assert e.value.status == aa.AA_ERR_ORDER and "aa_run_sps" in e.value.message
            seen.append(aa.aa_run_sps(g.h))
        assert seen == [aa.AA_STATUS_CHUNK_DONE] * (n - 1) + [aa.AA_STATUS_FINISHED]
        with pytest.raises(aa.AaError) as e:                               # after FINISHED: an error code, not a crash
            aa.aa_run_dedispersion(g.h, x)
        assert e.value.status == aa.AA_ERR_ORDER and "all" in e.value.message
        c1 = aa.aa_get_candidates(g.h)
        c2 = aa.aa_get_candidates(g.h)                                     # results stay valid and stable
        assert len(c1) == len(c2) > 0 and all(np.array_equal(c1[f], c2[f]) for f in c1.dtype.names)
        # immutable once configured: the description and geometry do not change by running
        assert aa.aa_strategy_describe(g.h) == desc0
        assert [aa.aa_strategy_get_range_info(g.h, r) for r in range(len(w.ranges))] == geo0
        # reset rewinds; a second run gives the same list
        aa.aa_strategy_reset(g.h)
        c3 = g.st.run(x)
        assert len(c3) == len(c1) and all(np.array_equal(c3[f], c1[f]) for f in c1.dtype.names)
    finally:
        g.close()


def test_candidate_overflow_is_counted_not_crashed():
    import paper_1912_07704_b200 as aa
    w = scaled(datagen.get_workload("tiny"), threshold=2.5, name="tiny_low_threshold")   # thousands of noise peaks
    x, _ = make_input(w)
    full = GpuRun(w, x, max_candidates=1 << 20)
    try:
        ref = full.st.run(x)
    finally:
        full.close()
    assert len(ref) > 500
    g = GpuRun(w, x, max_candidates=100)
    try:
        g.dedisperse()
        g.sps()
        with pytest.raises(aa.AaError) as e:
            aa.aa_get_candidates(g.h)
        assert e.value.status == aa.AA_ERR_CANDIDATE_OVERFLOW and str(len(ref)) in e.value.message   # the true count
        part = aa.aa_get_candidates(g.h, allow_overflow=True)
        assert len(part) == 100
        keys = set(zip(ref["range"].tolist(), ref["dm_index"].tolist(), ref["sample"].tolist()))
        assert all(k in keys for k in zip(part["range"].tolist(), part["dm_index"].tolist(), part["sample"].tolist()))
    finally:
        g.close()


@pytest.mark.parametrize("kind", ["quiet_head", "loud_head", "heavy_tails", "two_level"])
def test_row_statistics_fallback_routes_match_the_oracle(kind):
    """K3 reads a row once, using a core interval estimated from the row's first 8192 samples. These inputs break that
    estimate on purpose (head much quieter / much louder than the row, > 2.4 % outliers, bimodal row), forcing the list
    overflow and the 'bound cuts into the core' exits into the plain multi-pass route. mu and sigma must still equal the
    oracle's exactly, and so must the candidates."""
    rs = np.random.default_rng(99)
    C, N = 16, 70_000
    sig = np.full(N, 12.0)
    if kind == "quiet_head":
        sig[:12_000] = 0.7
    elif kind == "loud_head":
        sig[:12_000] = 60.0
    v = 127.0 + rs.standard_normal((C, N)) * sig
    if kind == "heavy_tails":
        m = rs.random((C, N)) < 0.06
        v[m] += rs.choice([-90.0, 90.0], size=int(m.sum()))
    if kind == "two_level":
        v[:, N // 2:] += 40.0
    x = np.clip(np.floor(v + 0.5), 0, 255).astype(np.uint8)
    w = Workload(kind, C, 1500.0, -1.0, 256e-6, N, ((0.0, 2.0, 6, 1), (12.0, 4.0, 5, 2)), (1, 2, 4, 8), 5.0, seed=1, npulses=0,
                 pulse_dm=(0.0, 0.0), pulse_width_max=1)
    gpu, orc = GpuRun(w, x), OracleRun(w, x)
    try:
        gpu.dedisperse()
        gpu.sps()
        exp = [check_band(gpu, orc, gpu.chunks[0], r, 0, rng[2], after_sps=True) for r, rng in enumerate(w.ranges)]
        compare_candidates(gpu.candidates(allow_overflow=True), np.concatenate(exp), w.threshold)
    finally:
        gpu.close()


@pytest.mark.parametrize("kind", ["gaussian_sparse", "uniform_dense", "mixed_groups"])
def test_offset_uint8_route_and_its_uint16_fallback_are_bit_exact(kind):
    """Binned ranges with bin 2 / 4 run K2 on bytes lo = clamp(x_b - off_c, 0, 255) plus an exactly scattered exception
    list; a channel group with too many exceptions takes the uint16 route instead (each kernel of both routes tests the
    same device counter). Inputs: Gaussian noise (few exceptions), uniform random bytes (about half the binned samples are
    exceptions: dense route), and channels 0..255 Gaussian / the rest uniform with >= 256 channels so that the channel
    groups of the pipelined copy choose DIFFERENT routes for the same chunk. Every row must equal the oracle's."""
    rs = np.random.default_rng(2024)
    C, N = (320, 12_000) if kind == "mixed_groups" else (24, 40_000)
    gauss = np.clip(np.floor(127.0 + 16.0 * rs.standard_normal((C, N)) + 0.5), 0, 255).astype(np.uint8)
    unif = rs.integers(0, 256, size=(C, N), dtype=np.uint8)
    if kind == "gaussian_sparse":
        x = gauss
    elif kind == "uniform_dense":
        x = unif
    else:
        x = np.where((np.arange(C) < 256)[:, None], gauss, unif).astype(np.uint8)
    nd = 2100 if kind != "mixed_groups" else 600            # many trials: a low exception limit (1e8 / ndms per group)
    w = Workload(kind, C, 1500.0, -0.5, 256e-6, N, ((0.0, 0.01, nd, 2), (30.0, 0.02, nd, 4)), (1, 2, 4), 6.0, seed=1, npulses=0,
                 pulse_dm=(0.0, 0.0), pulse_width_max=1)
    gpu, orc = GpuRun(w, x), OracleRun(w, x)
    try:
        assert "offset-uint8 route" in gpu.aa.aa_strategy_describe(gpu.h)
        gpu.dedisperse()
        chunk = gpu.chunks[0]
        for r, rng in enumerate(w.ranges):
            for (i0, i1) in ((0, 3), (nd // 2, nd // 2 + 3), (nd - 3, nd)):
                check_band(gpu, orc, chunk, r, i0, i1, after_sps=False)
        gpu.sps()
    finally:
        gpu.close()


def test_python_front_end_adds_no_appreciable_run_time():
    """PAPER.md:67 (§4): the Python front-end "did not show an appreciable runtime impact". The chunk loop driven from Python
    (two ctypes calls per chunk) against the same loop inside the library (aa_run_pipeline, one call): same candidates,
    and the wall-clock difference stays within a few per cent of a run that takes tens of milliseconds."""
    import time
    import torch
    import paper_1912_07704_b200 as aa
    w = scaled(datagen.get_workload("mid"), nsamp=1 << 16, name="mid64k")
    x, pinned = make_input(w, pinned=True)
    g = GpuRun(w, x, chunk_len_hint=16384)
    try:
        assert g.info["nchunks"] >= 5

        def python_loop():
            aa.aa_strategy_reset(g.h)
            return g.st.run(x)

        def c_loop():
            aa.aa_strategy_reset(g.h)
            assert aa.aa_run_pipeline(g.h, x) == aa.AA_STATUS_FINISHED
            return aa.aa_get_candidates(g.h)

        def best(f, n=7):
            ts = []
            for _ in range(n):
                torch.cuda.synchronize()
                t0 = time.perf_counter()
                c = f()
                torch.cuda.synchronize()
                ts.append(time.perf_counter() - t0)
            return min(ts), c

        python_loop(); c_loop()
        tp, cp = best(python_loop)
        tc, cc = best(c_loop)
        assert len(cp) == len(cc) > 0 and all(np.array_equal(cp[f], cc[f]) for f in cp.dtype.names)
        print(f"python loop {tp * 1e3:.3f} ms, C loop {tc * 1e3:.3f} ms, difference {100 * (tp - tc) / tc:+.2f} %")
        assert tp <= tc * 1.05 + 0.5e-3
    finally:
        g.close()


def test_boxcar_complete_chunks_match_the_oracle_and_recover_a_straddling_pulse():
    """Reading C3x (aa_plan_set_boxcar_overlap): rows are dedispersed E = W_max - 1 samples beyond the chunk's output span.
    Every row (incl. the extra samples), statistic and candidate equals the oracle's with the same E; the geometry is the
    oracle's; and a wide pulse placed across a chunk boundary, which the plain chunking only sees with narrow boxcars at
    the end of the chunk, is now found at its full width."""
    import oracle
    base = datagen.get_workload("tiny")
    widths = (1, 2, 4, 8, 16, 32, 64)
    E = max(widths) - 1
    L = 2048
    k = oracle.delay_constants(base.freqs_mhz, base.tsamp_s)
    geo = oracle.chunk_geometry(k, base.ranges, base.nsamp, chunk_len=L, boxcar_extra=E)
    t_edge = geo["chunks"][1][0] + geo["n_out"]                    # first output sample of chunk 2
    w = scaled(base, name="tiny_c3x", widths=widths, ranges=((0.0, 1.0, 60, 1), (60.0, 2.0, 20, 2)),
               fixed_pulses=((20.0, t_edge - 24, 48, 3.0),))        # 48 samples wide, half of it beyond the chunk's span
    x, _ = make_input(w)
    k = oracle.delay_constants(w.freqs_mhz, w.tsamp_s)
    geo = oracle.chunk_geometry(k, w.ranges, w.nsamp, chunk_len=L, boxcar_extra=E)
    gpu, orc = GpuRun(w, x, boxcar_overlap=True, chunk_len_hint=L), OracleRun(w, x)
    plain = GpuRun(w, x, chunk_len_hint=L)
    try:
        assert (gpu.info["overlap"], gpu.info["n_out"]) == (geo["S"], geo["n_out"]) and gpu.chunks == geo["chunks"]
        assert gpu.info["overlap"] > plain.info["overlap"]
        assert all(gpu.aa.aa_strategy_get_range_info(gpu.h, r)["boxcar_extra"] == E for r in range(len(w.ranges)))
        exp_all = []
        for chunk in gpu.chunks:
            gpu.dedisperse()
            gpu.sps()
            for r, rng in enumerate(w.ranges):
                exp_all.append(check_band(gpu, orc, chunk, r, 0, rng[2], after_sps=True))
        got = gpu.candidates()
        n, og, oe = compare_candidates(got, np.concatenate(exp_all), w.threshold)
        assert n + og == len(got) and n + oe == sum(len(e) for e in exp_all)
        # the straddling pulse: with C3x a candidate of width >= 32 starts within the last 48 samples before the edge
        near = (got["range"] == 0) & (got["sample"] >= t_edge - 48) & (got["sample"] < t_edge)
        assert near.any() and int(got["width"][near].max()) >= 32
        ref = plain.st.run(x)
        pe = plain.info["n_out"]                                    # the plain run's own chunk edges
        edges = [(j + 1) * pe for j in range(plain.info["nchunks"] - 1)]
        for e in edges:                                              # plain chunking: no boxcar can cross its chunk's end
            m = (ref["range"] == 0) & (ref["sample"] < e) & (ref["sample"] + ref["width"] > e)
            assert not m.any()
        assert ((got["range"] == 0) & (got["sample"] < t_edge) & (got["sample"] + got["width"] > t_edge)).any()
    finally:
        gpu.close()
        plain.close()


def test_clusters_of_the_tiny_pulse():
    """Reading C10 on real output: the injected pulse of the Tiny config produces ~20 candidates along its bow-tie in the
    (DM, time) plane; linked with a 2-DM-step / 8-sample tolerance the ones around the pulse merge into a cluster whose representative is
    the pulse itself, and the library's clusters equal the oracle's written-out definition on the same list."""
    import oracle
    w = datagen.get_workload("tiny")
    x, _ = make_input(w)
    g = GpuRun(w, x)
    try:
        cands = g.st.run(x)
        cl = g.aa.aa_get_clusters(g.h, 2.0, 8)
        clusters, reps = oracle.cluster_candidates(cands, 2.0, 8)
        assert len(cl) == len(clusters) and int(cl["members"].sum()) == len(cands)
        top = cl[np.argmax(cl["best"]["snr"])]
        assert int(top["members"]) >= 2 and len(cl) < len(cands)
        assert abs(int(top["best"]["dm_index"]) - 50) <= 1 and abs(int(top["best"]["sample"]) - 3000) <= 1 and int(top["best"]["width"]) == 4
        assert sorted(int(cands["sample"][r]) for r in reps) == sorted(int(s) for s in cl["best"]["sample"])
    finally:
        g.close()


@pytest.mark.parametrize("seed", range(int(__import__("os").environ.get("AA_TEST_FUZZ", "6"))))
def test_random_small_configurations_match_the_oracle(seed):
    """Randomised shapes and options (channel counts around the tile and group sizes, 1-3 DM ranges with random binning,
    arbitrary width lists, chunking, time-major input, boxcar-complete chunks, uniform or Gaussian samples, 8- or 16-bit input): every row,
    statistic and candidate equals the oracle's. AA_TEST_FUZZ=N runs N seeds (default 6)."""
    rs = np.random.default_rng(1000 + seed)
    C = int(rs.choice([1, 3, 7, 8, 9, 31, 64, 100, 255, 256, 257, 300, 520]))
    nr = int(rs.integers(1, 4))
    ranges, dm = [], 0.0
    for _ in range(nr):
        b = int(rs.choice([1, 2, 4, 8]))
        nd = int(rs.choice([1, 2, 29, 30, 31, 32, 33, 61, 64]))
        step = float(rs.choice([0.25, 0.5, 1.0, 3.0]))
        ranges.append((dm, step, nd, b))
        dm += step * nd
    widths = tuple(sorted(set(int(v) for v in rs.choice([1, 2, 3, 4, 5, 8, 16, 21, 32], size=int(rs.integers(1, 6)), replace=False))))
    tsamp = float(rs.choice([64e-6, 256e-6, 1024e-6]))
    f_top, bw = float(rs.choice([1500.0, 800.0, 420.0])), float(rs.choice([50.0, 100.0, 200.0]))
    B = max(r[3] for r in ranges)
    wtmp = Workload("fz", C, f_top, -bw / max(C, 2), tsamp, 1 << 20, tuple(ranges), widths, 5.0, seed=seed, npulses=0, pulse_dm=(0.0, 0.0), pulse_width_max=1)
    import oracle
    k = oracle.delay_constants(wtmp.freqs_mhz, tsamp)
    boxcar = bool(rs.integers(0, 2))
    E = (max(widths) - 1) if boxcar else 0
    S = oracle.chunk_geometry(k, ranges, 1 << 20, boxcar_extra=E)["S"]
    n_out_target = int(rs.choice([700, 2000, 5000])) * B
    nsamp = int(S + n_out_target * float(rs.choice([1.0, 2.6])) + int(rs.integers(0, 17)))
    if S > 300_000 or nsamp * C > 60_000_000:
        pytest.skip("delay span too large for a quick case")
    hint = 0
    if rs.integers(0, 2):
        hint = int(-(-(S + n_out_target) // B) * B)
        if hint >= (nsamp // B) * B:
            hint = 0
    bits16 = bool(rs.integers(0, 3) == 0)                                 # a third of the cases: 16-bit input samples
    depth = int(rs.choice([1023, 4095, 8191])) if bits16 else 255
    w = Workload("fz", C, f_top, -bw / max(C, 2), tsamp, nsamp, tuple(ranges), widths, 5.0, seed=seed, npulses=2, pulse_dm=(0.0, max(dm, 1.0)),
                 pulse_width_max=max(widths), pulse_snr=(9.0, 20.0), noise_mean=float(depth // 2) if bits16 else 127.0,
                 input_bits=16 if bits16 else 8, max_value=depth)
    x, _ = make_input(w)
    if rs.integers(0, 3) == 0:
        x = rs.integers(0, depth + 1, size=x.shape, dtype=x.dtype)        # dense exceptions: the dense route of every offset form
    tm = bool(rs.integers(0, 2))
    kw = dict(chunk_len_hint=hint) if hint else {}
    gpu, orc = GpuRun(w, x, time_major=tm, boxcar_overlap=boxcar, **kw), OracleRun(w, x)
    try:
        exp_all = []
        for j, chunk in enumerate(gpu.chunks):
            gpu.dedisperse()
            gpu.sps()
            for r, rng in enumerate(w.ranges):
                exp_all.append(check_band(gpu, orc, chunk, r, 0, rng[2], after_sps=True))
        got = gpu.candidates(allow_overflow=True)
        exp = np.concatenate(exp_all)
        if len(exp) < (1 << 20):
            n, og, oe = compare_candidates(got, exp, w.threshold)
            assert n + og == len(got) and n + oe == len(exp)
    finally:
        gpu.close()


def test_range_whose_tile_window_exceeds_shared_memory_takes_the_global_memory_route():
    """A DM step so coarse for the band that the 30 trials of a tile spread over more samples than shared memory holds is
    not a configuration error: the range runs the one-thread-per-output kernel on a device delay table (also in channel
    groups and next to ordinary ranges), with the same results as the oracle."""
    w = Workload("coarse", 272, 420.0, -200.0 / 272, 64e-6, 420_000, ((0.0, 40.0, 9, 1), (0.0, 0.05, 35, 2), (360.0, 20.0, 3, 8)),
                 (1, 2, 4, 8), 5.5, seed=12, npulses=2, pulse_dm=(0.0, 300.0), pulse_width_max=8, pulse_snr=(10.0, 20.0))
    x, _ = make_input(w)
    gpu, orc = GpuRun(w, x), OracleRun(w, x)
    try:
        assert "one-thread-per-output" in gpu.aa.aa_strategy_describe(gpu.h)
        gpu.dedisperse()
        gpu.sps()
        exp = [check_band(gpu, orc, gpu.chunks[0], r, 0, rng[2], after_sps=True) for r, rng in enumerate(w.ranges)]
        got = gpu.candidates()
        n, og, oe = compare_candidates(got, np.concatenate(exp), w.threshold)
        assert n + og == len(got) and n + oe == sum(len(e) for e in exp)
    finally:
        gpu.close()


@pytest.mark.parametrize("bits", [8, 16])
def test_sparse_exceptions_in_every_offset_form_are_scattered_exactly(bits):
    """Gaussian noise with rare large spikes (3e-5 of the samples, both signs) in a plan with bin 1, 2, 4 and 8: every offset
    form stays on its sparse route (exception rate below 4e-4) but has real exceptions with residuals of both signs - the
    offset-uint8 forms, the half-byte form with its bit plane (8-bit plans) and the offset-uint16 form (16-bit plans). Every row
    of D must equal the oracle's, in one chunk and with the channel groups of the pipelined copy (>= 256 channels)."""
    rs = np.random.default_rng(88 + bits)
    C, N = 288, 24_000
    mean, top = (127.0, 255) if bits == 8 else (1800.0, 4095)
    x = np.clip(np.floor(mean + 16.0 * rs.standard_normal((C, N)) + 0.5), 0, top)
    spikes = rs.random((C, N)) < 3e-5                               # bin 8: 2.4e-4 of the binned samples, below the 4e-4 route limit
    x[spikes] = np.where(rs.random(int(spikes.sum())) < 0.5, 0, top)
    x = x.astype(np.uint16 if bits == 16 else np.uint8)
    nd = 70
    w = Workload("spikes", C, 1500.0, -0.5, 256e-6, N, ((0.0, 0.05, nd, 1), (3.5, 0.05, nd, 2), (7.0, 0.1, nd, 4), (14.0, 0.2, nd, 8)), (1, 2, 4), 6.0,
                 seed=1, npulses=0, pulse_dm=(0.0, 0.0), pulse_width_max=1, input_bits=bits, max_value=top)
    gpu, orc = GpuRun(w, x), OracleRun(w, x)
    try:
        desc = gpu.aa.aa_strategy_describe(gpu.h)
        assert ("half-byte form" in desc) == (bits == 8) and ("offset-uint16 form" in desc) == (bits == 16)
        gpu.dedisperse()
        for r, rng in enumerate(w.ranges):
            check_band(gpu, orc, gpu.chunks[0], r, 0, nd, after_sps=False)
        gpu.sps()
        exp = [check_band(gpu, orc, gpu.chunks[0], r, 0, nd, after_sps=True) for r in range(len(w.ranges))]
        n, og, oe = compare_candidates(gpu.candidates(allow_overflow=True), np.concatenate(exp), w.threshold)
    finally:
        gpu.close()
