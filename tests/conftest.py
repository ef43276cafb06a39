import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")
    config.addinivalue_line("markers", "slow: long-running oracle check")


def pytest_collection_modifyitems(config, items):
    if os.environ.get("FG_RUN_SLOW"):
        return
    skip = pytest.mark.skip(reason="long-running oracle check: set FG_RUN_SLOW=1")
    for it in items:
        if "slow" in it.keywords:
            it.add_marker(skip)


def golden(name):
    return os.path.join(ROOT, "tests", "golden", name)


def read_facts():
    facts = {}
    with open(golden("paper_facts.txt")) as f:
        for line in f:
            line = line.split("#")[0].strip()
            if line:
                k, *v = line.split()
                facts[k] = v
    return facts
