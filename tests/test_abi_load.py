"""CPU-side checks of the boundary: libhisq.so builds, loads and exports every symbol include/hisq.h declares;
host-side index maps agree with the oracle's independent implementation.  No GPU compute here."""
import ctypes
import os
import re

import numpy as np
import pytest

import oracle
from paper_2306_01098_b200 import build as hisq_build
from paper_2306_01098_b200 import binding, layout

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    hisq_build.build()
    return binding.load_library()


def test_header_symbols_are_exported(lib):
    text = open(os.path.join(ROOT, "include", "hisq.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    declared = set(re.findall(r"\b(hisq_[A-Za-z_0-9]+)\s*\(", text))
    # the dynamic symbol table of the built library, not a list kept in Python: an export the header does not
    # declare (or the reverse) fails here
    import subprocess
    nm = subprocess.run(["nm", "-D", "--defined-only", binding.LIB_PATH], capture_output=True, text=True, check=True).stdout
    exported = {ln.split()[-1] for ln in nm.splitlines() if ln.split() and ln.split()[-1].startswith("hisq_")}
    assert declared == exported, declared ^ exported
    assert declared == set(binding.EXPORTS), declared ^ set(binding.EXPORTS)
    for name in declared:
        assert hasattr(lib, name), name


def test_strerror_and_invalid_create(lib):
    assert lib.hisq_strerror(0) == b"success"
    assert b"invalid" in lib.hisq_strerror(-1)
    h = ctypes.c_void_p()
    # odd extent, extent < 4, bad precision: rejected before any CUDA call
    assert lib.hisq_create(ctypes.byref(h), 7, 8, 8, 8, 8) == -1
    assert lib.hisq_create(ctypes.byref(h), 8, 8, 2, 8, 8) == -1
    assert lib.hisq_create(ctypes.byref(h), 8, 8, 8, 8, 5) == -1
    assert lib.hisq_workspace_bytes(None, 1) == 0


def test_sass_is_sm100a_and_has_vector_loads():
    import subprocess
    out = subprocess.run(["cuobjdump", "-lelf", binding.LIB_PATH], capture_output=True, text=True).stdout
    assert "sm_100a" in out


@pytest.mark.parametrize("L", [(4, 4, 4, 4), (8, 6, 4, 10), (6, 8, 8, 4), (12, 4, 6, 8)])
def test_product_index_maps_match_oracle(L):
    a = layout.eo_of_lex(L).numpy()
    assert np.array_equal(a, oracle.eo_index(L))
    inv = layout.lex_of_eo(L).numpy()
    assert np.array_equal(a[inv], np.arange(a.size))


def test_layout_rejects_bad_extents():
    for L in [(5, 4, 4, 4), (4, 4, 4, 2), (4, 4, 4)]:
        with pytest.raises(ValueError):
            layout.check_extents(L)
