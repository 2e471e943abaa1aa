"""The C-ABI library loads and exports every symbol include/mcdtn.h declares
(no compute calls: this runs without a GPU)."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "mcdtn.h")


def declared_functions():
    src = open(HEADER).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    names = re.findall(r"\b(mcs_[a-z0-9_]+)\s*\(", src)
    return sorted(set(names))


def test_header_declares_the_three_named_calls():
    names = declared_functions()
    for want in ("mcs_build_bvh", "mcs_estimate_dtn_interior", "mcs_estimate_dtn_exterior",
                 "mcs_closest_point", "mcs_free_bvh", "mcs_workspace_bytes", "mcs_error_string"):
        assert want in names


def test_library_exports_every_declared_symbol():
    from paper_2606_05581_b200.build import build
    lib = ctypes.CDLL(build())
    missing = [n for n in declared_functions() if not hasattr(lib, n)]
    assert not missing, missing
    lib.mcs_error_string.restype = ctypes.c_char_p
    lib.mcs_version.restype = ctypes.c_char_p
    assert lib.mcs_error_string(0) == b"ok"
    assert b"invalid" in lib.mcs_error_string(-1)
    assert b"sm_100a" in lib.mcs_version()


def test_binding_struct_sizes_match_header():
    """ctypes mirrors in api.py against sizes the compiler reports."""
    from paper_2606_05581_b200 import api
    from paper_2606_05581_b200.build import build
    lib = ctypes.CDLL(build())
    lib.mcs_abi_sizeof.restype = ctypes.c_size_t
    for which, cls in ((0, api._Samples), (1, api._Basis), (2, api._Params), (3, api._Matrix), (4, api.Stats), (5, api.BvhInfo),
                       (7, api._HostCoo), (8, api._BatchItem)):
        assert lib.mcs_abi_sizeof(ctypes.c_int(which)) == ctypes.sizeof(cls), cls.__name__


def test_no_cpu_fallback_in_binding():
    """The product path must fail loudly without the CUDA library / device."""
    import numpy as np
    import torch
    from paper_2606_05581_b200 import api
    with pytest.raises(ValueError):
        api.build_bvh(torch.zeros((3, 3)), torch.zeros((1, 3), dtype=torch.int32))   # CPU tensors rejected
    src = open(os.path.join(ROOT, "paper_2606_05581_b200", "api.py")).read()
    assert "oracle" not in src.replace("oracle-", "")
    assert np is not None
