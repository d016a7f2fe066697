import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)
sys.path.insert(0, os.path.dirname(os.path.abspath(__file__)))


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box via gpurun)")


def pytest_collection_modifyitems(config, items):
    try:
        import torch
        has_gpu = torch.cuda.is_available()
    except Exception:
        has_gpu = False
    if has_gpu:
        return
    skip = pytest.mark.skip(reason="no CUDA device")
    for item in items:
        if "gpu" in item.keywords:
            item.add_marker(skip)


def pytest_terminal_summary(terminalreporter):
    """Worst |d| / tolerance of every GPU-vs-oracle comparison of the run (test_gpu_parity.assert_parity)."""
    mod = sys.modules.get("test_gpu_parity")
    margins = getattr(mod, "MARGINS", None)
    if not margins:
        return
    worst = {}
    for test_id, rm, re_, n in margins:
        m = worst.setdefault(test_id, [0.0, 0.0, 0])
        m[0], m[1], m[2] = max(m[0], rm), max(m[1], re_), m[2] + n
    terminalreporter.write_sep("-", "parity margins: worst |d| / tolerance per test (mean, stderr, points compared)")
    for test_id, (rm, re_, n) in sorted(worst.items(), key=lambda kv: -max(kv[1][0], kv[1][1])):
        terminalreporter.write_line(f"{max(rm, re_):9.3e}  mean {rm:9.3e}  stderr {re_:9.3e}  {n:>10d}  {test_id}")
