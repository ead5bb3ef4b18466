"""CPU-only tests of the boundary and the host logic (run with -m "not gpu", no CUDA device needed):
  * libaa.so loads and exports every entry point include/aa.h declares, and the Python binding covers each of them;
  * plan validation gives an error code plus a message naming the field ("provides user feedback");
  * the strategy's host-side planning (delays, overlap, chunk list, per-range geometry) equals the oracle's geometry
    and the golden values of SURVEY §8(d); a planned-only strategy is NOT ready and refuses to run;
  * status codes are the ones the header states.
No compute call is made here.
"""
import re
from pathlib import Path

import numpy as np
import pytest

import datagen
import oracle
import paper_1912_07704_b200 as aa

ROOT = Path(__file__).resolve().parent.parent
HEADER = (ROOT / "include" / "aa.h").read_text()


def _declared_functions():
    # every "aa_xxx(" that is declared at the start of a line with a return type, i.e. the exported entry points
    names = re.findall(r"^(?:aa_status|void|size_t|const char\*)\s+(aa_[a-z0-9_]+)\s*\(", HEADER, flags=re.M)
    assert len(names) >= 20
    return sorted(set(names))


def test_library_exports_every_declared_symbol():
    lib = aa.load()
    for name in _declared_functions():
        assert hasattr(lib, name), f"libaa.so does not export {name} declared in include/aa.h"
        assert hasattr(aa, name), f"the Python binding has no function named {name}"
    assert "sm_100a" in aa.aa_version()


def test_status_codes_match_header():
    for name, value in re.findall(r"\b(AA_[A-Z_]+)\s*=\s*(-?\d+)", HEADER):
        assert getattr(aa, name) == int(value), name


def _plan(w):
    return aa.aa_plan_create(w.freqs_mhz, w.tsamp_s, w.ranges, w.widths, w.threshold)


@pytest.mark.parametrize("mutate,field", [
    (dict(freqs=np.array([1500.0, 1500.0, 1499.0])), "chan_freq"),          # not strictly descending
    (dict(freqs=np.array([], dtype=np.float64)), "nchans"),
    (dict(tsamp=0.0), "tsamp"),
    (dict(ranges=((0.0, 1.0, 10, 3),)), "bin"),                             # bin not in {1,2,4,8}
    (dict(ranges=((0.0, 1.0, 0, 1),)), "ndms"),
    (dict(ranges=((0.0, -1.0, 5, 1),)), "dm_step"),
    (dict(ranges=()), "nranges"),
    (dict(widths=(1, 4, 2)), "width"),                                      # not ascending
    (dict(widths=(0, 1)), "width"),
    (dict(widths=()), "nwidths"),
])
def test_plan_validation_names_the_field(mutate, field):
    w = datagen.get_workload("tiny")
    args = dict(freqs=w.freqs_mhz, tsamp=w.tsamp_s, ranges=w.ranges, widths=w.widths)
    args.update(mutate)
    with pytest.raises(aa.AaError) as e:
        aa.aa_plan_create(args["freqs"], args["tsamp"], args["ranges"], args["widths"], 6.0)
    assert e.value.status == aa.AA_ERR_INVALID_ARG
    assert field in str(e.value), str(e.value)


def test_plan_rejects_sums_that_would_overflow_the_packed_accumulators():
    freqs = 1500.0 - 0.01 * np.arange(40000)
    with pytest.raises(aa.AaError) as e:
        aa.aa_plan_create(freqs, 64e-6, ((0.0, 1.0, 4, 8),), (1,), 6.0)
    assert e.value.status == aa.AA_ERR_INVALID_ARG


def _golden_geometry():
    rows = {}
    for line in (ROOT / "tests" / "golden" / "geometry.txt").read_text().splitlines():
        if line.strip() and not line.startswith("#"):
            name, B, S, n_out, outputs = line.split()
            rows[name] = (int(B), int(S), int(n_out), int(outputs))
    return rows


@pytest.mark.parametrize("name", ["tiny", "mid", "ska", "lowf"])
def test_strategy_plan_geometry_equals_golden_and_oracle(name):
    w = datagen.get_workload(name)
    B, S, n_out, outputs = _golden_geometry()[name]
    plan = _plan(w)
    st = aa.aa_strategy_plan(plan, w.nsamp)
    try:
        info = aa.aa_strategy_get_info(st)
        assert info["ready"] == 0                                         # planned only: inspection, not execution
        assert (info["max_bin"], info["overlap"], info["n_out"], info["nchunks"]) == (B, S, n_out, 1)
        k = oracle.delay_constants(w.freqs_mhz, w.tsamp_s)
        g = oracle.chunk_geometry(k, w.ranges, w.nsamp)
        assert (g["S"], g["n_out"], g["L"]) == (info["overlap"], info["n_out"], info["chunk_len"])
        total = 0
        for r, rng in enumerate(w.ranges):
            ri = aa.aa_strategy_get_range_info(st, r)
            assert (ri["ndms"], ri["bin"], ri["nt"]) == (rng[2], rng[3], n_out // rng[3])
            assert ri["row_pitch"] >= ri["nt"]
            assert ri["max_delay"] == oracle.delay(k[-1], oracle.dm_value(rng[0], rng[1], rng[2] - 1), rng[3])
            total += ri["ndms"] * ri["nt"]
        assert total == outputs
        # the strategy's delay table is the oracle's, on a scatter of (range, dm, channel)
        rs = np.random.default_rng(5)
        for _ in range(200):
            r = int(rs.integers(len(w.ranges)))
            rng = w.ranges[r]
            i, c = int(rs.integers(rng[2])), int(rs.integers(w.nchans))
            assert aa.aa_strategy_get_delay(st, r, i, c) == oracle.delay(k[c], oracle.dm_value(rng[0], rng[1], i), rng[3])
        assert "chunk" in aa.aa_strategy_describe(st)
    finally:
        aa.aa_strategy_destroy(st)
        aa.aa_plan_destroy(plan)


def test_golden_delays_through_the_strategy():
    for line in (ROOT / "tests" / "golden" / "delays.txt").read_text().splitlines():
        if not line.strip() or line.startswith("#"):
            continue
        name, c, dm, b, d = line.split()
        w = datagen.get_workload(name)
        # a one-row plan at exactly this DM and bin
        plan = aa.aa_plan_create(w.freqs_mhz, w.tsamp_s, ((float(dm), 1.0, 1, int(b)),), (1,), 6.0)
        st = aa.aa_strategy_plan(plan, 1 << 21)
        try:
            assert aa.aa_strategy_get_delay(st, 0, 0, int(c)) == int(d), line
        finally:
            aa.aa_strategy_destroy(st)
            aa.aa_plan_destroy(plan)


def test_streaming_strategy_under_40gb_budget_tiles_the_time_axis():
    """BASELINE.json config 5: 600 s under a 40 GB budget -> overlapping chunks, overlap = max delay (rounded up to B)."""
    w = datagen.get_workload("stream")
    plan = _plan(w)
    st = aa.aa_strategy_plan(plan, w.nsamp, budget_bytes=40 * 10**9)
    try:
        info = aa.aa_strategy_get_info(st)
        assert info["overlap"] == 32384 and info["max_bin"] == 8
        assert info["arena_bytes_used"] <= 40 * 10**9
        assert info["nchunks"] >= 2 and info["chunk_len"] % 8 == 0 and info["chunk_len"] > info["overlap"]
        k = oracle.delay_constants(w.freqs_mhz, w.tsamp_s)
        g = oracle.chunk_geometry(k, w.ranges, w.nsamp, chunk_len=info["chunk_len"])
        assert len(g["chunks"]) == info["nchunks"]
        pos = 0
        for j in range(info["nchunks"]):
            start, length, n_out = aa.aa_strategy_get_chunk(st, j)
            assert (start, length, n_out) == tuple(g["chunks"][j])
            assert start == pos and start % 8 == 0 and length % 8 == 0 and n_out == length - info["overlap"]
            assert start + length <= w.nsamp
            pos += n_out
        assert w.nsamp - (pos + info["overlap"]) < 8                       # only a sub-bin tail is left over
    finally:
        aa.aa_strategy_destroy(st)
        aa.aa_plan_destroy(plan)


def test_budget_too_small_is_an_error_not_a_crash():
    w = datagen.get_workload("ska")
    plan = _plan(w)
    try:
        with pytest.raises(aa.AaError) as e:
            aa.aa_strategy_plan(plan, w.nsamp, budget_bytes=64 << 20)
        assert e.value.status == aa.AA_ERR_BUDGET_TOO_SMALL
        with pytest.raises(aa.AaError) as e:                             # input shorter than the maximum delay
            aa.aa_strategy_plan(plan, 30000)
        assert e.value.status in (aa.AA_ERR_INVALID_ARG, aa.AA_ERR_BUDGET_TOO_SMALL)
    finally:
        aa.aa_plan_destroy(plan)


def test_planned_only_strategy_refuses_to_run():
    """the API tells the user what still needs configuration; running before setup is NOT_READY."""
    w = datagen.get_workload("tiny")
    plan = _plan(w)
    st = aa.aa_strategy_plan(plan, w.nsamp)
    x = np.zeros((w.nchans, w.nsamp), np.uint8)
    try:
        for call in (lambda: aa.aa_run_dedispersion(st, x), lambda: aa.aa_run_sps(st), lambda: aa.aa_get_candidates(st)):
            with pytest.raises(aa.AaError) as e:
                call()
            assert e.value.status == aa.AA_ERR_NOT_READY
    finally:
        aa.aa_strategy_destroy(st)
        aa.aa_plan_destroy(plan)


def test_null_arguments_are_rejected():
    lib = aa.load()
    errs = (aa.AA_ERR_INVALID_ARG, aa.AA_ERR_NOT_READY)
    assert lib.aa_run_sps(None) in errs
    assert lib.aa_run_dedispersion(None, None, 0) in errs
    assert lib.aa_strategy_reset(None) in errs
    assert aa.aa_last_error() != ""
    lib.aa_plan_destroy(None)          # destroying NULL is a no-op (graceful exit)
    lib.aa_strategy_destroy(None)


def test_header_is_plain_c_and_links_from_c(tmp_path):
    """The boundary is a C ABI (no C++ in the header): a C99 translation unit that includes include/aa.h compiles with
    -Wall -Werror -pedantic, links against libaa.so and gets the documented error feedback without touching a GPU."""
    import subprocess
    src = tmp_path / "use_aa.c"
    src.write_text(r'''
#include <stdio.h>
#include <string.h>
#include "aa.h"
int main(void) {
    aa_plan* plan = NULL;
    double f[3] = {1500.0, 1499.0, 1498.0};
    aa_dm_range r = {0.0, 1.0, 4, 2};
    int32_t w[2] = {1, 2};
    if (aa_plan_create(&plan, 3, f, 64e-6, &r, 1, w, 2, 6.0f) != AA_OK) return 1;
    if (aa_plan_set_input_layout(plan, AA_LAYOUT_TIME_MAJOR) != AA_OK) return 2;
    if (aa_plan_set_input_layout(plan, 5) != AA_ERR_INVALID_ARG || !strstr(aa_last_error(), "layout")) return 3;
    aa_strategy* st = NULL;
    if (aa_strategy_plan(&st, plan, 4096, 0, 16, 0) != AA_OK) return 4;
    aa_strategy_info info;
    if (aa_strategy_get_info(st, &info) != AA_OK || info.ready != 0 || info.max_bin != 2 || info.input_layout != AA_LAYOUT_TIME_MAJOR) return 5;
    if (aa_run_sps(st) != AA_ERR_NOT_READY) return 6;
    r.bin = 3;
    aa_plan* bad = NULL;
    if (aa_plan_create(&bad, 3, f, 64e-6, &r, 1, w, 2, 6.0f) != AA_ERR_INVALID_ARG || !strstr(aa_last_error(), "bin")) return 7;
    aa_strategy_destroy(st);
    aa_plan_destroy(plan);
    printf("%s\n", aa_version());
    return 0;
}
''')
    exe = tmp_path / "use_aa"
    libdir = aa.lib_path().parent
    subprocess.check_call(["gcc", "-std=c99", "-Wall", "-Werror", "-pedantic", f"-I{ROOT / 'include'}", str(src), "-o", str(exe),
                           f"-L{libdir}", "-l:libaa.so", f"-Wl,-rpath,{libdir}"])
    out = subprocess.run([str(exe)], capture_output=True, text=True)
    assert out.returncode == 0, (out.returncode, out.stdout, out.stderr)
    assert "sm_100a" in out.stdout


# ------------------------------------------------------------------------------------------------ 16-bit plans
def test_input_bits_validation_names_the_limit_and_the_strategy_plans_the_offset_forms():
    """aa_plan_set_input_bits: the stated limits are checked with a message naming them; a 16-bit SKA-like plan has the same
    geometry as the 8-bit one (the sample type changes nothing in C2/C3), one more raw byte per sample in the arena, and
    every range on an offset form with the global-memory kernel behind it."""
    w = datagen.get_workload("ska16")
    plan = _plan(w)
    try:
        for bits, mx, word in ((12, 4095, "bits"), (16, 70000, "16 bits"), (16, 8192, "binned sample"), (16, 65535, "binned sample")):
            with pytest.raises(aa.AaError) as e:
                aa.aa_plan_set_input_bits(plan, bits, mx)
            assert e.value.status == aa.AA_ERR_INVALID_ARG and word in e.value.message, e.value.message
        aa.aa_plan_set_input_bits(plan, 16, w.max_value)
        st = aa.aa_strategy_plan(plan, w.nsamp)
        try:
            info = aa.aa_strategy_get_info(st)
            assert (info["input_bits"], info["input_max"], info["overlap"], info["n_out"], info["nchunks"]) == (16, 4095, 32384, 491904, 1)
            desc = aa.aa_strategy_describe(st)
            assert desc.count("offset-uint8 route") == 4 and "offset-uint16 form" in desc and desc.count("plain binned samples") == 5
            p8 = _plan(datagen.get_workload("ska"))
            s8 = aa.aa_strategy_plan(p8, w.nsamp)
            i8 = aa.aa_strategy_get_info(s8)
            aa.aa_strategy_destroy(s8); aa.aa_plan_destroy(p8)
            grow = info["arena_bytes_used"] - i8["arena_bytes_used"]
            assert 0.9 * w.nchans * w.nsamp < grow < 1.3 * w.nchans * w.nsamp      # the raw chunk is twice as large; delay tables
        finally:
            aa.aa_strategy_destroy(st)
    finally:
        aa.aa_plan_destroy(plan)
    # nchans * max_value * max bin must fit int32
    big = aa.aa_plan_create(1500.0 - 0.01 * np.arange(40000), 64e-6, ((0.0, 1.0, 4, 1),), (1,), 6.0)
    try:
        with pytest.raises(aa.AaError) as e:
            aa.aa_plan_set_input_bits(big, 16, 65535)                      # 40000 * 65535 > 2^31
        assert "int32" in e.value.message
        # still fine with a smaller maximum
        aa.aa_plan_set_input_bits(big, 16, 1023)
        aa.aa_plan_set_input_bits(big, 8, 0)
    finally:
        aa.aa_plan_destroy(big)


def test_chunk_rows_stay_below_the_28_bit_sample_field_of_an_exception_record():
    """An observation longer than 2^28 samples is chunked even without a budget (exception records carry the sample index in
    28 bits); a chunk_len_hint beyond that is refused with a message."""
    plan = aa.aa_plan_create(np.array([1500.0, 1499.0]), 64e-6, ((0.0, 1.0, 4, 2),), (1, 2), 6.0)
    try:
        n = (1 << 28) + 4096
        st = aa.aa_strategy_plan(plan, n)
        try:
            info = aa.aa_strategy_get_info(st)
            assert info["nchunks"] >= 2 and info["chunk_len"] < (1 << 28) and info["chunk_len"] % 2 == 0
        finally:
            aa.aa_strategy_destroy(st)
        with pytest.raises(aa.AaError) as e:
            aa.aa_strategy_plan(plan, n, chunk_len_hint=(1 << 28) + 2)
        assert e.value.status == aa.AA_ERR_INVALID_ARG and "largest chunk" in e.value.message
    finally:
        aa.aa_plan_destroy(plan)


def test_bench_refuses_a_multi_gpu_request_it_cannot_honour():
    """`python bench.py --gpus N` started without torchrun spawns its N ranks itself; on a node with fewer devices it must exit
    non-zero saying why, never print an n_gpus: 1 line (VERDICT r02 missing 1). A --gpus that contradicts WORLD_SIZE is refused too."""
    import os
    import subprocess
    import sys
    import torch
    if torch.cuda.is_available() and torch.cuda.device_count() >= 2:
        pytest.skip("this node could really run 2 ranks")
    root = Path(__file__).resolve().parent.parent
    env = {k: v for k, v in os.environ.items() if k not in ("WORLD_SIZE", "RANK", "LOCAL_RANK")}
    r = subprocess.run([sys.executable, str(root / "bench.py"), "--gpus", "2"], capture_output=True, text=True, env=env, timeout=300)
    assert r.returncode != 0 and "needs 2 CUDA devices" in r.stderr and r.stdout.strip() == ""
    r = subprocess.run([sys.executable, str(root / "bench.py"), "--gpus", "1"], capture_output=True, text=True,
                       env=dict(env, WORLD_SIZE="2", RANK="0", LOCAL_RANK="0"), timeout=300)
    assert r.returncode != 0 and "WORLD_SIZE = 2" in r.stderr and r.stdout.strip() == ""
