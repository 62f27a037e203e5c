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


@pytest.fixture(scope="session")
def built_library():
    """libkappagen.so is built in-tree (nvcc cross-compiles without a GPU); a no-op when it is up to date."""
    from paper_2602_05606_b200 import build as kbuild
    return kbuild.build()


# modules that pin the oracle and never touch the CUDA library: they must run on a box without nvcc
ORACLE_ONLY = {"test_oracle_cells", "test_oracle_direction", "test_oracle_distribution", "test_oracle_inverse",
               "test_oracle_literal", "test_oracle_params", "test_oracle_philox", "test_oracle_positions", "test_oracle_u64",
               "test_oracle_sanitizers"}


@pytest.fixture(autouse=True)
def _library_for_product_tests(request):
    if request.module.__name__.rsplit(".", 1)[-1] not in ORACLE_ONLY:
        request.getfixturevalue("built_library")
