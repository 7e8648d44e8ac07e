import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
# the library pipelines wm_score_topk_host by chunks of at least this many candidates (default 16384): a small value
# makes the chunked path run on the small batches of the tests; it must be set before libwm.so is first used
os.environ.setdefault("WM_HOST_CHUNK_MIN", "1024")
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box via gpurun)")


def read_golden(name):
    """Parse tests/golden/<name>: '#' comments, then 'key v0 v1 ...' lines -> dict of float lists."""
    out = {}
    with open(os.path.join(ROOT, "tests", "golden", name)) as f:
        for line in f:
            line = line.strip()
            if not line or line.startswith("#"):
                continue
            parts = line.split()
            out.setdefault(parts[0], []).append([float(x) for x in parts[1:]])
    return {k: (v[0] if len(v) == 1 else v) for k, v in out.items()}


@pytest.fixture(scope="session")
def golden():
    return read_golden
