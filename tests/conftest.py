import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


@pytest.fixture(scope="session")
def orc():
    import oracle
    oracle.build()
    return oracle


@pytest.fixture(scope="session")
def orc_rounding_variant(tmp_path_factory):
    """The oracle's own source rebuilt with different rounding: FMA contraction on (when the host CPU has FMA)
    and every sin / cos result moved by -1, 0 or +1 ulp (tests/jitter_trig.h).  It is still the oracle — the same
    algorithm, no CUDA — and measures how far two correct implementations of the map may differ."""
    from util import load_oracle_variant
    flags = ["-include", os.path.join(ROOT, "tests", "jitter_trig.h")]
    try:
        if " fma " in open("/proc/cpuinfo").read():
            flags += ["-ffp-contract=fast", "-mfma"]
    except OSError:
        pass
    return load_oracle_variant("rounding", flags, tmp_path_factory.mktemp("oracle_variant"))
