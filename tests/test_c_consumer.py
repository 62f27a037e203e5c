"""include/kappagen.h consumed from C: tests/c_abi/consumer.c is compiled with gcc -std=c99 against the header, linked
with libkappagen.so and the CUDA runtime, and run -- the argument-error contract on any box, one kappagen_sample checked
against oracle values on a GPU box (the boundary is a C ABI)."""
import os
import subprocess

import numpy as np
import pytest

import oracle
from gpu_util import TOL

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
PKG = os.path.join(ROOT, "paper_2602_05606_b200")
CUDA = os.environ.get("CUDA_HOME", "/usr/local/cuda")


@pytest.fixture(scope="module")
def consumer(tmp_path_factory, built_library):
    exe = str(tmp_path_factory.mktemp("c_abi") / "consumer")
    cmd = ["gcc", "-std=c99", "-pedantic", "-Wall", "-Wextra", "-Werror", "-O1", "-I", os.path.join(ROOT, "include"),
           "-isystem", os.path.join(CUDA, "include"), os.path.join(ROOT, "tests", "c_abi", "consumer.c"), "-o", exe,
           "-L", PKG, "-lkappagen", "-L", os.path.join(CUDA, "lib64"), "-lcudart", "-lm",
           "-Wl,-rpath," + PKG, "-Wl,-rpath," + os.path.join(CUDA, "lib64")]
    subprocess.run(cmd, check=True)
    return exe


def test_c_consumer_sees_the_documented_errors(consumer):
    r = subprocess.run([consumer, "errors"], capture_output=True, text=True, timeout=120)
    assert r.returncode == 0 and "errors ok" in r.stdout, (r.returncode, r.stdout, r.stderr)


@pytest.mark.gpu
@pytest.mark.parametrize("dtype", ["f32", "f64"])
def test_c_consumer_samples_what_the_oracle_computes(consumer, dtype):
    n, kappa, theta, seed, offset = 5000, 3.0, 0.7, 21, 2**32 - 1234
    want = oracle.sample(n, kappa, theta, seed, offset)
    args = [consumer, "sample", "0" if dtype == "f32" else "1", str(n), repr(kappa), repr(theta), str(seed), str(offset)]
    for i in (0, 1233, 1234, 4999):                           # both sides of the 2^32 counter carry, first and last
        args += [str(i)] + [repr(float(want[q][i])) for q in range(3)] + [repr(TOL[dtype])]
    r = subprocess.run(args, capture_output=True, text=True, timeout=300)
    assert r.returncode == 0 and "sample ok" in r.stdout, (r.returncode, r.stdout, r.stderr)
