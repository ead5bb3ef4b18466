"""aa_row_moments_static against aa_get_row_moments (GPU).

aa_row_moments_static is the library's one entry point for callers that cannot allocate device memory: a back-end whose
GPU memory is already divided up between its stages (a new cudaMalloc may fail, and the budget forbids it), or a watchdog
thread that must not freeze the streaming loop with the device-wide synchronisation every cudaMalloc / cudaFree implies.
Its working memory is a 256 KiB array built into libaa.so, shared by every call on a GPU and never cleared between calls
except by the calls themselves.

What is checked: the sums it returns for the rows of a dedispersed chunk equal those of the existing, arena-backed path
(aa_get_row_moments) exactly - both are integer sums, so the bar is equality as everywhere else in this suite - on two
calls in a row whose row counts and row lengths differ, so that the second call would show any sums the first one left
behind in the shared array. The size limit is checked to be refused with a message, before anything is launched.

This file sorts last on purpose (pytest -x stops at the first failure: a failure here must not hide the parity tests), and
it sets up its own strategy so that it passes alone in a fresh process as well as after the rest of the suite.
"""
import numpy as np
import pytest

import datagen
from datagen.workloads import scaled

from helpers import GpuRun, make_input

pytestmark = pytest.mark.gpu


def _two_range_workload():
    """Tiny's band with two DM ranges of different length and binning: 101 rows of about 69 900 samples (five ragged
    slices per row in the sliced kernel) and 37 rows of about 34 950 (three)."""
    w = datagen.get_workload("tiny")
    return scaled(w, nsamp=70016, name="tiny-two-ranges", ranges=((0.0, 1.0, 101, 1), (101.0, 2.0, 37, 2)))


def test_static_moments_equal_the_arena_path_on_two_calls_in_a_row():
    w = _two_range_workload()
    x, _ = make_input(w)
    gpu = GpuRun(w, x)
    aa = gpu.aa
    try:
        gpu.dedisperse()
        aa.aa_synchronize(gpu.h)
        chunk_n_out = gpu.chunks[0][2]
        expected, got = [], []
        for r in (0, 1):                                   # existing path first: it runs on the strategy's own stream
            expected.append(gpu.moments(r))
        for r in (0, 1):                                   # then the two calls under test, back to back
            ptr, pitch = aa.aa_get_dedispersed_device(gpu.h, r)
            nt = chunk_n_out // w.ranges[r][3]
            got.append(aa.aa_row_moments_static(ptr, pitch, nt, w.ranges[r][2]))
        for r in (0, 1):
            assert got[r][0].shape == (w.ranges[r][2],)
            assert np.array_equal(got[r][0], expected[r][0]), f"range {r}: sum_t D differs from aa_get_row_moments"
            assert np.array_equal(got[r][1], expected[r][1]), f"range {r}: sum_t t*D differs from aa_get_row_moments"
        assert np.any(expected[0][0] != 0) and np.any(expected[1][1] != 0)     # the comparison is not 0 == 0

        # the same call again, and a shorter slice of range 0 (fewer rows AND fewer samples than the call before it):
        # every word this call uses still holds the larger sums of the previous one until the call clears it
        ptr, pitch = aa.aa_get_dedispersed_device(gpu.h, 0)
        again = aa.aa_row_moments_static(ptr, pitch, chunk_n_out, w.ranges[0][2])
        assert np.array_equal(again[0], expected[0][0]) and np.array_equal(again[1], expected[0][1])
        head = aa.aa_row_moments_static(ptr, pitch, 1000, 5)
        rows = np.stack([gpu.row(0, i)[:1000].astype(np.int64) for i in range(5)])
        assert np.array_equal(head[0], rows.sum(axis=1))
        assert np.array_equal(head[1], (rows * np.arange(1000, dtype=np.int64)).sum(axis=1))
    finally:
        gpu.close()


def test_static_moments_refuse_more_rows_than_the_built_in_array_holds():
    import paper_1912_07704_b200 as aa
    import torch
    d = torch.zeros(16, dtype=torch.int32, device="cuda")
    with pytest.raises(aa.AaError) as err:
        aa.aa_row_moments_static(d, 0, 0, aa.AA_STATIC_MOMENTS_MAX_ROWS + 1)
    assert err.value.status == aa.AA_ERR_INVALID_ARG and str(aa.AA_STATIC_MOMENTS_MAX_ROWS) in str(err.value)
    a, b = aa.aa_row_moments_static(d, 16, 16, 0)          # no rows: nothing to do, not an error
    assert a.size == 0 and b.size == 0
