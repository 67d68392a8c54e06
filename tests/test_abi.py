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


def test_struct_layouts_match_header(tmp_path):
    """sizeof / offsetof of the two ABI structs as a C compiler sees include/lqcd.h (gcc, no CUDA needed)
    against the ctypes mirrors in the binding."""
    import subprocess
    from paper_1109_2935_b200 import lqcd
    src = tmp_path / "layout.c"
    src.write_text('''#include <stdio.h>
#include <stddef.h>
#include "lqcd.h"
int main(void) {
  printf("%zu %zu %zu %zu %zu %zu %zu\\n", sizeof(lqcd_invert_params), sizeof(lqcd_invert_result),
         offsetof(lqcd_invert_params, schwarz_block), offsetof(lqcd_invert_params, mr_omega),
         offsetof(lqcd_invert_params, matpc_type), offsetof(lqcd_invert_result, true_residual),
         offsetof(lqcd_invert_result, gflop));
  return 0;
}
''')
    exe = tmp_path / "layout"
    subprocess.check_call(["gcc", "-I", os.path.join(ROOT, "include"), "-o", str(exe), str(src)])
    got = [int(t) for t in subprocess.check_output([str(exe)], text=True).split()]
    want = [ctypes.sizeof(lqcd.InvertParams), ctypes.sizeof(lqcd.InvertResult), lqcd.InvertParams.schwarz_block.offset,
            lqcd.InvertParams.mr_omega.offset, lqcd.InvertParams.matpc_type.offset, lqcd.InvertResult.true_residual.offset,
            lqcd.InvertResult.gflop.offset]
    assert got == want


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
