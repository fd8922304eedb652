"""CPU-side checks of the boundary: the C-ABI library builds for sm_100a, loads, and exports every
symbol include/tkm.h declares; host-only entry points (folds, argument validation) behave.  No
compute call is made (there is no GPU here)."""
import ctypes
import os
import re

import numpy as np
import pytest

import oracle as o

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def tkm():
    from paper_2606_06742_b200 import build
    build.build()
    import paper_2606_06742_b200 as t
    t.lib()
    return t


def _declared_symbols():
    txt = open(os.path.join(ROOT, "include", "tkm.h")).read()
    txt = re.sub(r"/\*.*?\*/", "", txt, flags=re.S)
    return sorted(set(re.findall(r"\b(tkm_[a-z0-9_]+)\s*\(", txt)))


def test_library_exports_every_declared_symbol(tkm):
    names = _declared_symbols()
    assert {"tkm_gram", "tkm_spectral_setup", "tkm_fit_path", "tkm_exact_cv", "tkm_predict"} <= set(names)
    L = ctypes.CDLL(tkm.lib_path())
    for nme in names:
        assert hasattr(L, nme), "libtkm.so does not export %s" % nme
    assert sorted(tkm.EXPORTED_SYMBOLS) == names
    assert tkm.tkm_version() == 1


def test_no_alloc_limit_of_the_binding_is_the_header_constant(tkm):
    from paper_2606_06742_b200.api import PREDICT_NOALLOC_MAX_COEF
    txt = open(os.path.join(ROOT, "include", "tkm.h")).read()
    m = re.search(r"#define\s+TKM_PREDICT_NOALLOC_MAX_COEF\s+(\d+)", txt)
    assert m and int(m.group(1)) == PREDICT_NOALLOC_MAX_COEF == 65536


def test_sass_has_fp64_tensor_core_and_tma_instructions(tkm):
    import subprocess
    out = subprocess.run(["cuobjdump", "-sass", tkm.lib_path()], capture_output=True, text=True).stdout
    assert "DMMA" in out and "sm_100a" in out
    assert "UTMALDG" in out      # operand tiles of the contractions are staged by TMA


@pytest.mark.parametrize("n,V,seed", [(200, 5, 7), (17, 4, 0), (1001, 10, 2**63 + 5), (2000, 5, 7)])
def test_make_folds_bit_exact_with_oracle(tkm, n, V, seed):
    assert np.array_equal(tkm.tkm_make_folds(n, V, seed), o.make_folds(n, V, seed))


def test_make_folds_rejects_bad_arguments(tkm):
    with pytest.raises(tkm.TkmError) as e:
        tkm.tkm_make_folds(3, 5, 1)
    assert e.value.code == 1 and "V" in str(e.value)


def test_missing_library_fails_loudly(tkm, monkeypatch):
    import paper_2606_06742_b200.api as api
    monkeypatch.setattr(api, "_lib", None)
    monkeypatch.setattr(api, "lib_path", lambda: "/nonexistent/libtkm.so")
    with pytest.raises(api.TkmError):
        api.lib()
