"""Seeded synthetic inputs shared by the oracle-side tests and the CUDA path.

This package holds no arithmetic of the search method: ``dg.c`` draws
noise and stamps pulses whose per-channel offsets are handed in as data; ``workloads.py`` holds the
five BASELINE.json configurations (frequencies, DM plans, widths, thresholds, pulse draws) and the
signal model used to sweep an injected pulse across the band.
"""
from .generator import build, generate, checksum, lib_path  # noqa: F401
from .workloads import WORKLOADS, Workload, get_workload, pulse_sweep, scaled  # noqa: F401
