"""The C-ABI library loads and exports every symbol include/kappagen.h declares; host-only entry points
and argument checks behave as documented.  No kernel is launched here (CPU box)."""
import ctypes
import os
import re

import pytest

import oracle
from paper_2602_05606_b200 import build as kbuild
from paper_2602_05606_b200 import kappagen as kg

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def L():
    kbuild.build()
    return kg.lib()


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "kappagen.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(kappagen_[a-z_0-9]+)\s*\(", text)))


def test_every_declared_symbol_is_exported(L):
    names = declared_symbols()
    assert len(names) >= 18 and "kappagen_words_tile" in names and "kappagen_velocity_of_words_tile" in names and "kappagen_speed_histogram" in names and "kappagen_sample_flags" in names and "kappagen_sample_cells_moments" in names and "kappagen_sample" in names and "kappagen_sample_cells" in names
    for name in names:
        assert getattr(L, name) is not None


def test_version_and_params_match_oracle(L):
    assert kg.version() >= 100
    for kappa in (1.6, 2.0, 3.0, 4.0, 6.0, 10.0, 15.0, 1000.0):
        got, want = kg.params(kappa), oracle.params(kappa)
        for g, w in zip(got, want):
            assert abs(g - w) <= 4e-16 * abs(w)


def test_argument_errors_are_reported_before_any_launch(L):
    for bad in (1.5, 1.0, float("nan"), float("inf")):
        with pytest.raises(kg.KappagenError) as e:
            kg.params(bad)
        assert e.value.status == kg.EINVAL
    f = L.kappagen_sample
    assert f(-1, 2.0, 1.0, 0, 0, kg.F32, None, None, None, None) == kg.EINVAL
    assert "negative" in kg.last_error()
    assert f(8, 2.0, 1.0, 0, 0, 7, 16, 16, 16, None) == kg.EINVAL            # bad dtype
    assert f(8, 2.0, 1.0, 0, 0, kg.F32, None, 16, 16, None) == kg.ENULL
    assert f(8, 2.0, 1.0, 0, 0, kg.F64, 16, 20, 16, None) == kg.EALIGN        # 20 is not 8-byte aligned
    assert f(8, 1.5, 1.0, 0, 0, kg.F32, 16, 16, 16, None) == kg.EINVAL        # kappa > 3/2 strictly
    assert f(8, 2.0, -1.0, 0, 0, kg.F32, 16, 16, 16, None) == kg.EINVAL
    assert f(0, 2.0, 1.0, 0, 0, kg.F32, None, None, None, None) == kg.OK      # n = 0: nothing to do
    g = L.kappagen_sample_cells
    assert g(4, 2, 16, 16, None, 0, 0, 0, kg.F32, 16, 16, 16, None, 0, None) == kg.EWORKSPACE
    assert g(4, 2, 16, 16, 16, 5, 0, 0, kg.F32, 16, 16, 16, 16, 1 << 20, None) == kg.EINVAL   # bad drift stride
    assert g(4, 2, None, 16, None, 0, 0, 0, kg.F32, 16, 16, 16, 16, 1 << 20, None) == kg.ENULL
    assert g(0, 64, None, None, None, 0, 0, 0, kg.F32, None, None, None, None, 0, None) == kg.OK
    assert L.kappagen_cells_workspace_bytes(10, kg.F32) == 10 * 48      # one 12-value record per cell
    assert L.kappagen_cells_workspace_bytes(10, kg.F64) == 10 * 96
    assert L.kappagen_words(-3, 0, 0, None, None, None, None) == kg.EINVAL
    assert L.kappagen_words(3, 0, 0, None, None, None, None) == kg.ENULL


def test_missing_library_fails_loudly(monkeypatch):
    monkeypatch.setattr(kg, "_lib", None)
    monkeypatch.setattr(kg, "_SO", "/nonexistent/libkappagen.so")
    with pytest.raises(kg.KappagenNotBuilt):
        kg.lib()


def test_product_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_2602_05606_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".cpp", ".hpp", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in text and "from oracle" not in text and "oracle/" not in text.replace("oracle/.", ""), f
