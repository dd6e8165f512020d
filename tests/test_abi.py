"""The C-ABI library builds, loads, and exports every symbol include/pd.h declares (no compute calls: no GPU here)."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def libpath():
    from paper_2006_09808_b200 import build
    return build.build()


def header_functions():
    src = open(os.path.join(ROOT, "include", "pd.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(pd_[a-z_]+)\s*\(", src)))


def test_header_and_binding_agree():
    from paper_2006_09808_b200 import binding
    assert header_functions() == sorted(binding.SYMBOLS)


def test_library_exports_every_declared_symbol(libpath):
    L = C.CDLL(libpath)
    for name in header_functions():
        assert hasattr(L, name), name


def test_error_paths_that_need_no_gpu(libpath):
    from paper_2006_09808_b200 import binding
    L = binding.lib()
    assert binding.strerror(binding.OK) == "success"
    assert "64, 128, 256, 512" in binding.strerror(binding.ESIZE)
    h = C.c_void_p()
    assert L.pd_plan(None, 64, 64, 1, 1, 0.01, 0.25, 0.25, 1.0) == binding.EINVAL
    assert L.pd_plan(C.byref(h), 64, 64, 0, 1, 0.01, 0.25, 0.25, 1.0) == binding.EINVAL        # batch < 1
    assert L.pd_plan(C.byref(h), 64, 64, 1, 7, 0.01, 0.25, 0.25, 1.0) == binding.EINVAL        # bad B0_dir
    assert L.pd_plan(C.byref(h), 64, 64, 1, 1, -1.0, 0.25, 0.25, 1.0) == binding.EINVAL        # lambda < 0
    assert L.pd_plan(C.byref(h), 64, 64, 1, 1, 0.01, 0.25, 0.25, 1.5) == binding.EINVAL        # theta > 1
    assert L.pd_plan(C.byref(h), 258, 256, 1, 1, 0.01, 0.25, 0.25, 1.0) == binding.ESIZE       # paper's 258: NEXT-1
    assert L.pd_plan(C.byref(h), 64, 100, 1, 1, 0.01, 0.25, 0.25, 1.0) == binding.ESIZE
    assert L.pd_plan(C.byref(h), 64, 64, 1, 1, 0.01, 0.4, 0.4, 1.0) == binding.ESTEP           # 0.16*8.44 > 1
    assert h.value is None
    assert L.pd_solve(None, None, None, None, 1, 0.0, None) == binding.EINVAL
    assert L.pd_destroy(None) == binding.EINVAL
    assert L.pd_set_option(None, 0, 0) == binding.EINVAL


def test_product_does_not_import_the_oracle():
    """The product path may not route through oracle/ (or any CPU fallback)."""
    pkg = os.path.join(ROOT, "paper_2006_09808_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "pd_oracle" not in text and "oracle/" not in text.replace("the CPU oracle", ""), f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".cpp", ".h", ".py")):
            text = open(os.path.join(ROOT, "oracle", f)).read()
            assert "#include \"../paper" not in text and "import paper_2006_09808_b200" not in text
            assert "csrc/" not in text.replace("paper_2006_09808_b200/csrc/", "")  # only mentioned in a comment
