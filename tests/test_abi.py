"""The C-ABI library (include/madme.h): builds, loads, exports every declared symbol, validates arguments and
refuses to compute without a CUDA device (there is no CPU path).  No GPU needed."""
import ctypes as C
import os
import re

import pytest
import torch

from paper_2211_14056_b200 import api, build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    build.build()
    return api.lib()


def _declared_functions():
    src = open(os.path.join(ROOT, "include", "madme.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"^\s*(?:const\s+)?(?:int|void|double|long long|char\s*\*)\s*\*?\s*(\w+)\s*\(", src, flags=re.M)))


def test_header_and_binding_agree():
    assert _declared_functions() == sorted(api.SYMBOLS)


def test_library_exports_every_declared_symbol(lib):
    for name in _declared_functions():
        assert hasattr(lib, name), name


def test_python_binding_has_the_same_names():
    for name in api.SYMBOLS:
        if name in ("me_last_error", "me_n_external", "me_n_final"):
            continue
        assert callable(getattr(api, name)), name


def test_argument_validation_without_compute(lib):
    out = C.c_void_p()
    p = api.MeParams(0.118, 1 / 132.507, 173.0, 0.0, 20.0, 0.4)
    assert lib.me_init(b"no_such_process", C.byref(p), C.byref(out)) == api.ME_EPROCESS
    assert b"no_such_process" in lib.me_last_error()
    assert lib.me_init(None, C.byref(p), C.byref(out)) == api.ME_EINVAL
    pw = api.MeParams(0.118, 1 / 132.507, 173.0, 1.5, 20.0, 0.4)
    assert lib.me_init(b"gg_ttx", C.byref(pw), C.byref(out)) == api.ME_EINVAL  # a width would break the closed form
    assert lib.philox_uniform(0, 0, 0, 8, None, 4, None) == api.ME_EINVAL
    assert lib.philox_uniform(0, 0, 0, 99, C.c_void_p(16), 4, None) == api.ME_EDIM
    m = (C.c_double * 2)(0.0, 0.0)
    assert lib.rambo_generate(C.c_void_p(16), 100.0, m, 9, 0, C.c_void_p(16), C.c_void_p(16), 4, None) == api.ME_EDIM
    assert lib.rambo_generate(C.c_void_p(16), 100.0, m, 2, 0, C.c_void_p(8), C.c_void_p(16), 4, None) == api.ME_EINVAL  # alignment
    heavy = (C.c_double * 2)(60.0, 60.0)
    assert lib.rambo_generate(C.c_void_p(16), 100.0, heavy, 2, 0, C.c_void_p(16), C.c_void_p(16), 4, None) == api.ME_EINVAL
    assert lib.me_eval(None, None, None, 0, None) == api.ME_EINVAL
    assert lib.vegas_iterate(None, None, 1000.0, 10, None, None) == api.ME_EINVAL


@pytest.mark.skipif(torch.cuda.is_available(), reason="checks the no-device behaviour")
def test_no_cpu_fallback(lib):
    """Without a CUDA device the product refuses: it never computes on the CPU."""
    out = C.c_void_p()
    p = api.MeParams(0.118, 1 / 132.507, 173.0, 0.0, 20.0, 0.4)
    assert lib.me_init(b"gg_ttx", C.byref(p), C.byref(out)) == api.ME_ENODEV
    assert lib.philox_uniform(0, 0, 0, 8, C.c_void_p(16), 4, None) == api.ME_ENODEV
    assert lib.vegas_unweight_static_init() == api.ME_ENODEV
    assert lib.vegas_unweight_static(C.c_void_p(16), 4, 1.0, 0, 0, 0, C.c_void_p(16), C.c_void_p(16), None) == api.ME_ENODEV
    with pytest.raises(api.MadmeError):
        api.me_init("gg_ttxgg", dict(alpha_s=0.118, alpha_em=1 / 132.507, m_top=173.0, w_top=0.0, ptj_min=20.0, dr_min=0.4))


def test_product_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_2211_14056_b200")
    for root, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".inc", ".h")):
                text = open(os.path.join(root, f)).read()
                assert "import oracle" not in text and "from oracle" not in text and "oracle/" not in text.replace("shares no source with oracle/", ""), f
