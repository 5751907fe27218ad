"""No GPU needed: the C-ABI library loads and exports every function include/ia.h declares; the
binding declares the same set; struct sizes match the header's layout."""
import ctypes
import os
import re

import pytest

from paper_2401_04576_b200 import binding as b

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    src = open(os.path.join(ROOT, "include", "ia.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(ia_[a-z0-9_]+)\s*\(", src)))


def test_header_declares_the_north_star_calls():
    names = _declared()
    for must in ("ia_load_geometry", "ia_vote", "ia_topk", "ia_refine", "ia_refine_batch"):
        assert must in names


def test_library_exports_every_declared_symbol():
    from paper_2401_04576_b200 import build
    lib = ctypes.CDLL(build.build())
    for name in _declared():
        assert hasattr(lib, name), f"{name} declared in ia.h but not exported"
    assert sorted(b.EXPORTS) == _declared()
    assert lib.ia_pad_ulps() == 4
    lib.ia_strerror.restype = ctypes.c_char_p
    assert lib.ia_strerror(-3).startswith(b"parameter box")


def test_struct_layouts():
    assert b.WIRE_DT.itemsize == 56 and b.HIT_DT.itemsize == 16 and b.BOX_DT.itemsize == 88
    assert ctypes.sizeof(b.IaParams) == 40
    assert b.BOX_DT.fields["votes"][1] == 80


def test_no_gpu_means_loud_failure():
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(RuntimeError):
        b.Context(0)
