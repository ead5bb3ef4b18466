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
        t = torch.empty((w.nchans, w.nsamp), dtype=torch.uint8, pin_memory=True)
        x = t.numpy()
        datagen.generate(w.seed, w.nchans, w.nsamp, pl, dl, out=x)
        return x, t
    return datagen.generate(w.seed, w.nchans, w.nsamp, pl, dl), None


class OracleRun:
    """Oracle-side view of one workload: delay constants and binned chunks (cached per (chunk, bin))."""

    def __init__(self, w, x):
        self.w, self.x = w, x
        self.k = oracle.delay_constants(w.freqs_mhz, w.tsamp_s)
        self._xb = {}

    def binned(self, start, length, b):
        key = (start, length, b)
        if key not in self._xb:
            self._xb = {k: v for k, v in self._xb.items() if k[:2] == (start, length)}   # keep one chunk's worth
            self._xb[key] = oracle.bin_time(self.x, start, length // b, b)
        return self._xb[key]

    def search(self, chunk, r_index, i0, i1, want=("D", "stats")):
        start, length, n_out = chunk
        rng = self.w.ranges[r_index]
        xb = self.binned(start, length, rng[3])
        return oracle.search_rows(xb, self.k, rng, r_index, n_out // rng[3], self.w.widths, self.w.threshold, start, i0, i1, want=want)


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
