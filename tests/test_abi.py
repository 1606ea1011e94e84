"""Host-side checks of the C-ABI boundary (no GPU needed): the library builds, loads, and exports
every function include/qcd.h declares; without a device it refuses to create a context."""
import ctypes

import numpy as np
import pytest

import paper_1710_09178_b200 as q
from paper_1710_09178_b200 import binding, build


@pytest.fixture(scope="module")
def lib():
    build.build()
    return q.load_library()


def test_header_symbols_all_exported(lib):
    names = q.exported_symbols()
    assert {"qcd_create", "qcd_destroy", "qcd_dslash", "qcd_mdagm", "qcd_multishift_cg", "qcd_load_gauge",
            "qcd_pack", "qcd_unpack", "qcd_dslash_host", "qcd_multishift_cg_host",
            "qcd_last_error"} <= set(names)
    for n in names:
        assert hasattr(lib, n), f"{n} declared in include/qcd.h but not exported"
    # the binding covers the whole header, nothing more
    assert set(binding._SIGNATURES) == set(names)


def test_version_string(lib):
    assert b"sm_100a" in lib.qcd_version()


def test_create_rejects_bad_dims_before_touching_cuda(lib):
    h = ctypes.c_void_p(None)
    for dims in [(3, 4, 4, 4), (4, 4, 4, 0), (4, 4, 1, 4), (4, 6, 4, -2)]:
        cd = (ctypes.c_int * 4)(*dims)
        st = lib.qcd_create(cd, 0.1, None, ctypes.byref(h))
        assert st == binding.QCD_EINVAL and not h.value
        assert b"even" in lib.qcd_last_error(None)
    assert lib.qcd_create(None, 0.1, None, ctypes.byref(h)) == binding.QCD_EINVAL
    assert lib.qcd_create((ctypes.c_int * 4)(4, 4, 4, 4), 0.1, None, None) == binding.QCD_EINVAL


def test_no_cpu_fallback_without_device(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    h = ctypes.c_void_p(None)
    st = lib.qcd_create((ctypes.c_int * 4)(4, 4, 4, 4), 0.1, None, ctypes.byref(h))
    assert st == binding.QCD_ECUDA and not h.value
    with pytest.raises(q.QcdError):
        q.Context((4, 4, 4, 4), 0.1, stream=0)


def test_null_context_is_an_error_not_a_crash(lib):
    assert lib.qcd_dslash(None, 0, None, None) == binding.QCD_EINVAL
    assert lib.qcd_mdagm(None, 0, None, None) == binding.QCD_EINVAL
    assert lib.qcd_destroy(None) == binding.QCD_OK
    assert lib.qcd_vector_doubles(None) == 0


def test_product_does_not_import_oracle():
    """The product path must not route through the oracle (nor the oracle through the product)."""
    import os
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    for sub, banned in (("paper_1710_09178_b200", "oracle"), ("oracle", "paper_1710_09178_b200"),
                        ("lattice_inputs", "oracle"), ("lattice_inputs", "paper_1710_09178_b200")):
        for dirpath, _, files in os.walk(os.path.join(root, sub)):
            for fn in files:
                if fn.endswith((".py", ".cu", ".cuh", ".c", ".h")):
                    text = open(os.path.join(dirpath, fn)).read()
                    for line in text.splitlines():
                        s = line.strip()
                        if s.startswith(("import ", "from ", "#include")):
                            assert banned not in s, f"{sub}/{fn}: {s}"
