import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")


@pytest.fixture(scope="session")
def cfg1_scene():
    import noit_scenes
    return noit_scenes.cfg1(0)


def pytest_terminal_summary(terminalreporter):
    """Largest |gpu - oracle| / (1e-5 max + 1e-6) seen by each parity test."""
    try:
        from test_parity_gpu import RATIOS
    except Exception:
        return
    if not RATIOS:
        return
    terminalreporter.write_line("parity: largest |gpu - oracle| / (1e-5 max(|a|,|b|) + 1e-6) per test")
    for k, v in sorted(RATIOS.items(), key=lambda kv: -kv[1])[:12]:
        terminalreporter.write_line(f"  {v:8.3f}  {k}")
