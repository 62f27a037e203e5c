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


@pytest.fixture(scope="session", autouse=True)
def built_library():
    """libkappagen.so is built in-tree (nvcc cross-compiles without a GPU); a no-op when it is up to date."""
    from paper_2602_05606_b200 import build as kbuild
    return kbuild.build()
