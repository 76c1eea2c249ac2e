"""CPU-side checks of the C-ABI library: it loads, exports every symbol include/hea.h declares, validates
arguments before touching a device, and fails loudly (HEA_ECUDA, no fallback) when there is no GPU."""
import ctypes as C
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def L():
    from paper_2411_18906_b200 import build
    build.build()
    from paper_2411_18906_b200 import binding
    return binding.lib()


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "hea.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(hea_[a-z_]+)\s*\(", text)))


def test_exports_every_declared_symbol(L):
    from paper_2411_18906_b200 import binding
    names = declared_symbols()
    assert len(names) >= 15
    assert sorted(binding.EXPORTS) == names
    for n in names:
        assert getattr(L, n) is not None
    assert b"sm_100a" in L.hea_version()


def test_argument_validation_precedes_device_use(L):
    h = C.c_void_p()
    conc = np.array([0.5, 0.5]); w = np.array([1.0]); t = np.zeros(4)
    p = lambda a: a.ctypes.data_as(C.c_void_p)
    assert L.hea_create(C.byref(h), 0, 2, 2, 2, 9, p(conc), 1, p(w), p(t), 0) == 2        # HEA_EUNSUPPORTED
    assert L.hea_create(C.byref(h), 0, 2, 2, 2, 2, p(conc), 4, p(w), p(t), 0) == 2
    assert L.hea_create(C.byref(h), 5, 2, 2, 2, 2, p(conc), 1, p(w), p(t), 0) == 1        # HEA_EINVAL
    assert L.hea_create(C.byref(h), 0, 0, 2, 2, 2, p(conc), 1, p(w), p(t), 0) == 1
    bad = np.array([0.5, 0.4])
    assert L.hea_create(C.byref(h), 0, 2, 2, 2, 2, p(bad), 1, p(w), p(t), 0) == 1
    assert b"sum to 1" in L.hea_last_error()
    assert L.hea_create(None, 0, 2, 2, 2, 2, p(conc), 1, p(w), p(t), 0) == 1
    assert L.hea_info(None, None, None, None) == 1
    assert L.hea_destroy(None) == 0
    # the ordered pair counts are int32: max_s(z_s) * N must stay below 2^31 (fcc 283^3 with three shells: 24 * 90.6e6)
    w3 = np.array([1.0, 0.5, 0.25]); t3 = np.zeros(12)
    assert L.hea_create(C.byref(h), 0, 283, 283, 283, 2, p(conc), 3, p(w3), p(t3), 0) == 2
    assert b"2^31" in L.hea_last_error()
    # non-finite weights and targets are argument errors
    assert L.hea_create(C.byref(h), 0, 2, 2, 2, 2, p(conc), 1, p(np.array([np.nan])), p(t), 0) == 1
    tinf = np.zeros(4); tinf[1] = np.inf
    assert L.hea_create(C.byref(h), 0, 2, 2, 2, 2, p(conc), 1, p(w), p(tinf), 0) == 1
    assert L.hea_measure_peaks(None, None, 0, None) == 1


def test_no_cpu_fallback_without_a_device(L):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    h = C.c_void_p()
    conc = np.array([0.5, 0.5]); w = np.array([1.0]); t = np.zeros(4)
    p = lambda a: a.ctypes.data_as(C.c_void_p)
    assert L.hea_create(C.byref(h), 1, 2, 2, 2, 2, p(conc), 1, p(w), p(t), 0) == 4        # HEA_ECUDA
    assert b"no CPU fallback" in L.hea_last_error()
    assert not h.value


def test_product_package_does_not_touch_the_oracle():
    pkg = os.path.join(ROOT, "paper_2411_18906_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".cpp", ".hpp", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "hea_oracle" not in src and "libhea_oracle" not in src, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c", ".h")):
            src = open(os.path.join(ROOT, "oracle", f)).read()
            assert "import paper_2411_18906_b200" not in src and "from paper_2411_18906_b200" not in src
            assert "hea.h" not in src and "libhea_b200" not in src
