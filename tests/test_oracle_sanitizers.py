"""The oracle under AddressSanitizer and UndefinedBehaviorSanitizer (the oracle is what every GPU
result is judged against, so an out-of-bounds read or a signed overflow in IT would be a silent error in the judge).
The C++ source is compiled a second time with -fsanitize=address,undefined (no recovery: the first finding aborts) and
every exported function is driven through oracle/__init__.py in a child process -- empty, single, ragged and
counter-carry sizes, the extreme words, invalid cells -- with the sanitizer runtime preloaded."""
import os
import subprocess
import sys
import textwrap

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

DRIVER = textwrap.dedent('''
    import sys
    import numpy as np
    sys.path.insert(0, sys.argv[2])
    import oracle
    oracle._SO = sys.argv[1]                 # the sanitised build (newer than the source: build() leaves it alone)
    assert oracle.lib()._name == sys.argv[1]
    edge = np.array([0, 1, 2, 0x7fffffff, 0x80000000, 0xfffffffe, 0xffffffff, 12345], dtype=np.uint32)
    oracle.philox4x32_10([0, 0, 0, 0], [0, 0])
    oracle.philox4x32_10([0xffffffff] * 4, [0xffffffff] * 2)
    for n, off in ((0, 0), (1, 0), (1001, 2**32 - 500), (257, 2**64 - 100)):
        oracle.words(n, 7, off)
        for kappa in (1.6, 4.1, 50.0):
            oracle.sample(n, kappa, 0.5, 7, off)
            oracle.sample(n, kappa, 0.0, 7, off, literal=True)
            oracle.sample_u64(n, kappa, 1.5, 7, off, return_w3=True)
            oracle.speed_over_theta(n, kappa, 7, off)
            oracle.speed_over_theta(n, kappa, 7, off, u64=True)
        oracle.positions(n, 7, off, 23)
        oracle.positions(n, 7, off, 32)
    for kappa in (1.5000001, 1.6, 2.0, 3.95, 4.6, 10.0, 1e4):
        oracle.params(kappa)
        oracle.x_of_w0(edge, kappa); oracle.x_of_w0_literal(edge, kappa); oracle.L_of_w0(edge, kappa)
        oracle.x_of_w0w3(edge, edge[::-1].copy(), kappa)
        oracle.velocity_of_words(edge, edge[::-1].copy(), edge, kappa, 2.0)
        oracle.velocity_of_words_u64(edge, edge, edge[::-1].copy(), edge, kappa, 2.0)
    oracle.direction(edge, edge[::-1].copy())
    kap = np.array([2.0, 1.5, np.nan, 3.0, np.inf, 5.0]); th = np.array([1.0, 1.0, 1.0, -1.0, 1.0, 0.0])
    drift = np.arange(18, dtype=np.float64) * 0.01
    for ppc in (0, 1, 5, 64):
        oracle.sample_cells(ppc, kap, th, None, 0, 3, 2**32 - 7)
        oracle.sample_cells(ppc, kap, th, drift[:3], 0, 3, 11, thermal=True)
        oracle.sample_cells(ppc, kap, th, drift, 1, 3, 11)
        oracle.cells_moments(ppc, kap, th, drift, 1, 3, 11)
    oracle.sample_cells(4, kap[:0], th[:0], None, 0, 3, 0)
    s = oracle.speed_over_theta(5000, 3.0, 1)
    h = oracle.speed_histogram(s, 0.2, 64)
    for which in ("exact", "approx"):
        oracle.bin_probabilities(3.0, 0.2, 64, which)
        oracle.relative_entropy(h, 3.0, 0.2, 1e-10, which)
    print("sanitised oracle: all calls returned")
''')


def test_oracle_is_clean_under_asan_and_ubsan(tmp_path):
    asan = subprocess.run(["gcc", "-print-file-name=libasan.so"], capture_output=True, text=True).stdout.strip()
    if not os.path.isabs(asan) or not os.path.exists(asan):
        pytest.skip("no libasan in this toolchain")
    so = str(tmp_path / "libkappagen_oracle_san.so")
    src = os.path.join(ROOT, "oracle", "kappagen_oracle.cpp")
    subprocess.run(["g++", "-std=c++17", "-O1", "-g", "-fPIC", "-shared", "-fsanitize=address,undefined",
                    "-fno-sanitize-recover=all", "-fno-omit-frame-pointer", "-o", so, src, "-lm"], check=True)
    drv = tmp_path / "drive.py"
    drv.write_text(DRIVER)
    env = dict(os.environ, LD_PRELOAD=asan, ASAN_OPTIONS="detect_leaks=0:abort_on_error=0:exitcode=23",
               UBSAN_OPTIONS="print_stacktrace=1:halt_on_error=1")
    r = subprocess.run([sys.executable, str(drv), so, ROOT], capture_output=True, text=True, env=env, timeout=600)
    assert r.returncode == 0, (r.returncode, r.stderr[-3000:])
    assert "all calls returned" in r.stdout
    assert "runtime error" not in r.stderr and "AddressSanitizer" not in r.stderr, r.stderr[-3000:]
