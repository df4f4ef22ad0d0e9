import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
for p in (ROOT, os.path.join(ROOT, "tests")):
    if p not in sys.path:
        sys.path.insert(0, p)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (B200); run with -m gpu")
    config.addinivalue_line("markers", "slow: long full-size parity runs (minutes of oracle time); opt in with "
                                       "SHASTA_SLOW=1 or -m 'gpu and slow'")


def pytest_collection_modifyitems(config, items):
    # the slow full-size runs stay out of the default `-m gpu` selection (the driver's round-end budget)
    if os.environ.get("SHASTA_SLOW") == "1" or "slow" in (config.getoption("-m") or ""):
        return
    skip = pytest.mark.skip(reason="slow: set SHASTA_SLOW=1 or select with -m 'gpu and slow'")
    for it in items:
        if "slow" in it.keywords:
            it.add_marker(skip)


def pytest_sessionfinish(session, exitstatus):
    """Achieved parity numbers (GPU vs oracle) of this session -> gpurun_out/parity_r2.json (merged with what a
    previous session wrote); profiles/parity_r2.json is a copy of it."""
    import json
    import parity
    if not parity._RECORD:
        return
    out = os.path.join(ROOT, "gpurun_out")
    os.makedirs(out, exist_ok=True)
    path = os.path.join(out, "parity_r2.json")
    data = {}
    if os.path.exists(path):
        try:
            data = json.load(open(path))
        except Exception:
            data = {}
    data.update(parity._RECORD)
    json.dump(data, open(path, "w"), indent=1, sort_keys=True)


@pytest.fixture(scope="session")
def oracle():
    from oracle import shasta_oracle as so
    so.build()
    so.set_threads(os.cpu_count() or 1)
    return so
