import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run with -m gpu on a B200)")


def read_facts():
    facts = {}
    with open(os.path.join(ROOT, "tests", "golden", "paper_printed_facts.txt")) as f:
        for line in f:
            line = line.split("#", 1)[0].strip()
            if line:
                k, v = line.split("=")
                facts[k.strip()] = float(v)
    return facts


@pytest.fixture(scope="session")
def facts():
    return read_facts()
