"""The five BASELINE.json configurations as data, plus the pulse draws.

Nothing here is part of the search: a Workload is the parameter set handed to ``aa_plan_create`` (and to
the oracle) together with the recipe of the synthetic input. ``pulse_sweep`` is the SIGNAL MODEL of an
injected pulse (cold-plasma dispersion law, t0 referred to the top channel), used only to place the
synthetic pulses; tests pin it against the oracle's own delay function.

Readings: frequencies f_c = f_top + c*foff with channel 0 the top of the band;
DM ranges half-open [lo, hi) with ndms = (hi-lo)/step; boxcar widths powers of two up to the stated
maximum; pulse amplitude A = snr * sigma_noise / sqrt(nchans * width) (white-noise matched-filter gain).
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

DISPERSION_CONSTANT = 4.148808e3  # s MHz^2 pc^-1 cm^3, BASELINE.json north_star


@dataclass(frozen=True)
class Workload:
    name: str
    nchans: int
    f_top_mhz: float
    foff_mhz: float
    tsamp_s: float
    nsamp: int
    ranges: tuple            # ((dm_low, dm_step, ndms, bin), ...)
    widths: tuple            # boxcar widths in binned samples, ascending
    threshold: float
    seed: int
    npulses: int
    pulse_dm: tuple          # (lo, hi) uniform
    pulse_width_max: int
    pulse_snr: tuple = (8.0, 20.0)
    fixed_pulses: tuple = ()  # ((dm, t0, width, amp), ...) overrides the random draw
    budget_bytes: int = 0     # 0 = no budget stated (single chunk)
    noise_mean: float = 127.0
    noise_sigma: float = 16.0
    input_bits: int = 8       # 8: uint8 samples; 16: uint16 samples clipped to [0, max_value]
    max_value: int = 255      # the largest sample value the telescope delivers (the stated bit depth)

    @property
    def dtype(self):
        return np.uint16 if self.input_bits == 16 else np.uint8

    @property
    def gen_kw(self) -> dict:
        """Keyword arguments of datagen.generate that this workload fixes (noise level, sample type)."""
        return dict(mean=self.noise_mean, sigma=self.noise_sigma, bits=self.input_bits, max_value=self.max_value)

    @property
    def freqs_mhz(self) -> np.ndarray:
        return self.f_top_mhz + np.arange(self.nchans, dtype=np.float64) * self.foff_mhz

    @property
    def ndms_total(self) -> int:
        return sum(r[2] for r in self.ranges)

    def pulses(self):
        """Return (list of (t0, width, amp), dms[np], delays int64 [np][nchans])."""
        f = self.freqs_mhz
        if self.fixed_pulses:
            dms = np.array([p[0] for p in self.fixed_pulses], dtype=np.float64)
            pl = [(int(p[1]), int(p[2]), float(p[3])) for p in self.fixed_pulses]
        else:
            rng = np.random.default_rng(self.seed)
            dms = rng.uniform(self.pulse_dm[0], self.pulse_dm[1], self.npulses)
            # widths log-uniform on 1..pulse_width_max, SNR uniform on pulse_snr
            wid = np.maximum(1, np.round(2.0 ** rng.uniform(0.0, np.log2(self.pulse_width_max), self.npulses))).astype(np.int64)
            snr = rng.uniform(self.pulse_snr[0], self.pulse_snr[1], self.npulses)
            amp = snr * self.noise_sigma / np.sqrt(self.nchans * wid.astype(np.float64))
            u = rng.uniform(0.0, 1.0, self.npulses)
            pl = []
            for i in range(self.npulses):
                sweep = int(pulse_sweep(f, dms[i], self.tsamp_s)[-1])
                room = max(1, self.nsamp - sweep - int(wid[i]) - 1)
                pl.append((int(u[i] * room), int(wid[i]), float(amp[i])))
        delays = np.stack([pulse_sweep(f, d, self.tsamp_s) for d in dms]) if len(dms) else np.zeros((0, self.nchans), np.int64)
        return pl, dms, delays


def pulse_sweep(freqs_mhz: np.ndarray, dm: float, tsamp_s: float) -> np.ndarray:
    """Arrival offset (samples, int64) of a pulse of dispersion measure ``dm`` in each channel relative to
    channel 0: nearest sample to DISPERSION_CONSTANT*dm*(f^-2 - f0^-2) seconds."""
    f = np.asarray(freqs_mhz, dtype=np.float64)
    dt = DISPERSION_CONSTANT * float(dm) * (1.0 / (f * f) - 1.0 / (f[0] * f[0]))
    return np.floor(dt / tsamp_s + 0.5).astype(np.int64)


def _pow2(wmax):
    return tuple(1 << k for k in range(wmax.bit_length()) if (1 << k) <= wmax)


_SKA_RANGES = ((0.0, 0.1, 1500, 1), (150.0, 0.2, 750, 1), (300.0, 0.25, 800, 2),
               (500.0, 0.4, 1000, 4), (900.0, 1.0, 1100, 8))

WORKLOADS = {
    "tiny": Workload("tiny", 64, 1500.0, -1.0, 256e-6, 8192, ((0.0, 1.0, 101, 1),), (1, 2, 4, 8, 16), 6.0,
                     1912, 1, (50.0, 50.0), 4, fixed_pulses=((50.0, 3000, 4, 12.0),)),
    "mid": Workload("mid", 1024, 1550.0, -300.0 / 1024, 64e-6, 1 << 18, ((0.0, 0.5, 1001, 1),), _pow2(64), 6.0,
                    7704, 20, (10.0, 500.0), 32),
    "ska": Workload("ska", 4096, 1500.0, -300.0 / 4096, 64e-6, 1 << 19, _SKA_RANGES, _pow2(256), 7.0,
                    20191207, 50, (0.0, 2000.0), 256),
    "lowf": Workload("lowf", 4096, 350.0, -150.0 / 4096, 64e-6, 1 << 21,
                     ((0.0, 0.05, 2000, 1), (100.0, 0.1, 1500, 2), (250.0, 0.1, 2500, 4)), _pow2(512), 7.0,
                     3500200, 100, (5.0, 500.0), 512),
    # the SKA-like configuration delivered as 16-bit samples of 12-bit depth (noise N(1800, 16), pulses as in ska)
    "ska16": Workload("ska16", 4096, 1500.0, -300.0 / 4096, 64e-6, 1 << 19, _SKA_RANGES, _pow2(256), 7.0,
                      20191207, 50, (0.0, 2000.0), 256, noise_mean=1800.0, input_bits=16, max_value=4095),
    "stream": Workload("stream", 4096, 1500.0, -300.0 / 4096, 64e-6, 9_375_000, _SKA_RANGES, _pow2(256), 7.0,
                       600, 300, (0.0, 2000.0), 256, budget_bytes=40 * 10**9),
}


def get_workload(name: str) -> Workload:
    return WORKLOADS[name]


def scaled(w: Workload, *, nsamp: int | None = None, name: str | None = None, **kw) -> Workload:
    """A copy of ``w`` with some fields replaced (parity tests use shorter streams of the same shape)."""
    from dataclasses import replace
    if nsamp is not None:
        kw["nsamp"] = nsamp
    if name is not None:
        kw["name"] = name
    return replace(w, **kw)
