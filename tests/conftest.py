import os
import sys
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parent.parent
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))


def _ensure_built():
    """The native pieces are built in-tree and git-ignored: build them if a fresh checkout has none (no-op when up to date).
    nvcc cross-compiles for sm_100a without a GPU."""
    from paper_1912_07704_b200 import build as aa_build
    aa_build.build(verbose=False)
    import datagen
    import oracle
    datagen.build()
    oracle.build()


def pytest_configure(config):
    _ensure_built()
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")
    config.addinivalue_line("markers", "slow: full-size configuration (minutes)")


@pytest.fixture(scope="session")
def tiny():
    """Tiny workload: (workload, x, k, geometry) generated once per session."""
    import datagen
    import oracle
    w = datagen.get_workload("tiny")
    pl, dms, dl = w.pulses()
    x = datagen.generate(w.seed, w.nchans, w.nsamp, pl, dl)
    k = oracle.delay_constants(w.freqs_mhz, w.tsamp_s)
    g = oracle.chunk_geometry(k, w.ranges, w.nsamp)
    return w, x, k, g
