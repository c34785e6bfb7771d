import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")
    config.addinivalue_line("markers", "slow: long-running CPU test")


@pytest.fixture(scope="session", autouse=True)
def _internal_guard_bands():
    """TM_DEBUG_GUARDS=1 runs the WHOLE GPU suite with sentinel margins around every internal device buffer of the library
    (tm_debug_guards, include/tm.h) and fails the session's last test if any margin was written to - the memcheck stand-in
    where compute-sanitizer cannot run (profiles/r02_guard_bands.md has the recorded run)."""
    if os.environ.get("TM_DEBUG_GUARDS") != "1":
        yield
        return
    import torch
    if not torch.cuda.is_available():
        yield
        return
    from paper_2107_09879_b200 import libtm
    libtm.debug_guards(1)
    yield
    bad, n = libtm.debug_guards(-1)
    print(f"\n[tm_debug_guards] guarded internal blocks: {n}, damaged margins: {bad}")
    assert bad == 0, f"{bad} damaged margin(s) around internal device buffers"
