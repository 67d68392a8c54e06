"""CPU-side checks (-m "not gpu"): the C-ABI library loads and exports every symbol that
include/lqcd.h declares; the binding's struct layouts match the header; the product never
imports the oracle.  No compute call is made (no GPU here)."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "lqcd.h")
LIB = os.path.join(ROOT, "paper_1109_2935_b200", "liblqcd_b200.so")


def _declared():
    src = open(HEADER).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(lqcd_[a-z_0-9]+)\s*\(", src)))


@pytest.fixture(scope="module")
def lib():
    if not os.path.exists(LIB):
        import __graft_entry__
        __graft_entry__.build()
    return ctypes.CDLL(LIB)


def test_every_declared_symbol_is_exported(lib):
    names = _declared()
    assert len(names) >= 18
    for n in names:
        assert hasattr(lib, n), n


def test_binding_lists_the_same_symbols():
    from paper_1109_2935_b200 import lqcd
    assert sorted(lqcd.EXPORTS) == _declared()


def test_struct_layouts_match_header():
    from paper_1109_2935_b200 import lqcd
    # lqcd_invert_params: 4 doubles, 10 ints, int[4], int, double, 2 ints  (natural alignment)
    assert ctypes.sizeof(lqcd.InvertParams) == 4 * 8 + 10 * 4 + 16 + 4 + 4 + 8 + 8
    assert ctypes.sizeof(lqcd.InvertResult) == 6 * 4 + 4 * 8
    assert lqcd.InvertParams.mr_omega.offset % 8 == 0


def test_create_without_gpu_fails_loudly(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    from paper_1109_2935_b200 import lqcd
    with pytest.raises(lqcd.LqcdError):
        lqcd.Context((4, 4, 4, 4), (1, 1, 1, -1), 0)


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_1109_2935_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt and "liboracle" not in txt, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".cpp")):
            txt = open(os.path.join(ROOT, "oracle", f)).read()
            assert "import paper_1109_2935_b200" not in txt and "from paper_1109_2935_b200" not in txt
            assert "lqcd.h" not in txt or f.endswith(".py")
