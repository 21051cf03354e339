import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run with -m gpu on a B200)")
    config.addinivalue_line("markers", "slow: long CPU pin, still part of the default CPU suite")


HOOKS = ["PRAND_MT_CFG", "PRAND_MT_APPLY", "PRAND_GM_LP", "PRAND_GM31_NF", "PRAND_GM_WATCH", "PRAND_MRG_INT",
         "PRAND_GM_INIT", "PRAND_CHUNK_LEN", "PRAND_LFSR_INIT", "PRAND_MT_POLY", "PRAND_SEQ_SECTIONS"]

import pytest  # noqa: E402


@pytest.fixture(autouse=True)
def _no_hook_outlives_its_test():
    """prand_debug_set changes a process-wide table: whatever a test forced (an alternate kernel, a chunk length) is
    cleared when the test ends, also when it fails, so that no later test runs on a path it did not ask for."""
    yield
    pkg = sys.modules.get("paper_1307_5869_b200")
    if pkg is not None and getattr(pkg, "_lib", None) is not None:
        for name in HOOKS:
            pkg._lib.prand_debug_set(name.encode(), None)
