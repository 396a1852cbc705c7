"""CPU-side checks of the C-ABI library: it builds for sm_100a, loads, exports every symbol that
include/lof.h declares, and validates parameters before touching a device."""
import ctypes as C
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lof():
    from paper_1701_08197_b200 import build, lof as m
    build.build_lib()
    return m


def _declared():
    src = open(os.path.join(ROOT, "include", "lof.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(lof_[a-z0-9_]+)\s*\(", src)))


def test_exports_match_header(lof):
    L = lof.lib()
    names = _declared()
    assert len(names) >= 12
    for n in names:
        assert hasattr(L, n), n
    assert sorted(lof.EXPORTS) == names


def test_struct_layout(lof):
    assert C.sizeof(lof.Params) == 60
    assert lof.STATS_DTYPE.itemsize == 32
    assert lof.STATS_DTYPE.fields["mean"][1] == 8 and lof.STATS_DTYPE.fields["n_flagged"][1] == 24


def test_factor_table_host(lof):
    f = lof.factor_table(10)
    want = np.array([6 * 0.75 ** k for k in range(10)])
    assert np.array_equal(f, want)             # exact in fp64 for p = 1.5 (6, 4.5)
    assert f[0] == 6.0 and f[1] == 4.5


@pytest.mark.parametrize("kw", [dict(S=0), dict(Cn=0), dict(T=0), dict(max_window=3), dict(max_window=2048),
                                dict(max_window=0), dict(directions=0), dict(directions=4), dict(p=0.0),
                                dict(sensitivity=-1.0), dict(start_threshold=float("nan")), dict(Cn=257),
                                dict(history_length=4, history_min_fill=0), dict(history_sensitivity=float("inf")),
                                dict(sir_eta=-0.1), dict(sir_eta=1.5), dict(sir_eta=float("nan")), dict(stats_mode=2)])
def test_bad_params_rejected_before_device(lof, kw):
    a = dict(S=1, Cn=4, T=64)
    a.update({k: v for k, v in kw.items() if k in a})
    rest = {k: v for k, v in kw.items() if k not in a}
    prm = lof.make_params(a["S"], a["Cn"], a["T"], **rest)
    h = C.c_void_p()
    assert lof.lib().lof_create(C.byref(prm), C.byref(h)) == lof.E_PARAM
    assert not h.value


def test_struct_size_and_null(lof):
    prm = lof.make_params(1, 4, 64)
    prm.struct_size = 8
    h = C.c_void_p()
    assert lof.lib().lof_create(C.byref(prm), C.byref(h)) == lof.E_PARAM
    assert lof.lib().lof_create(None, C.byref(h)) == lof.E_NULL
    assert lof.lib().lof_create(C.byref(prm), None) == lof.E_NULL
    assert lof.lib().lof_destroy(None) == 0
    assert b"parameter" in lof.lib().lof_strerror(lof.E_PARAM)


def test_no_cpu_fallback_without_device(lof):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a device is present")
    prm = lof.make_params(1, 4, 64)
    h = C.c_void_p()
    assert lof.lib().lof_create(C.byref(prm), C.byref(h)) == lof.E_CUDA      # fails loudly, no fallback
    with pytest.raises(lof.LofError):
        lof.Flagger(1, 4, 64)


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_1701_08197_b200")
    for dp, _, fs in os.walk(pkg):
        for f in fs:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dp, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt and "lof_oracle" not in txt, f
