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
    return sorted(set(re.findall(r"\b(pd_[a-z0-9_]+)\s*\(", src)))


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
    assert L.pd_plan(C.byref(h), 257, 256, 1, 1, 0.01, 0.25, 0.25, 1.0) == binding.ESIZE       # odd lengths are not supported
    assert L.pd_plan(C.byref(h), 64, 2, 1, 1, 0.01, 0.25, 0.25, 1.0) == binding.ESIZE
    assert L.pd_plan(C.byref(h), 2048, 64, 1, 1, 0.01, 0.25, 0.25, 1.0) == binding.ESIZE
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


def test_line_factors_host_logic(libpath):
    """pd_line_factors (pure host arithmetic): the tuned power-of-two lines, and the balanced two-factor split of the
    general-length kernels (the paper's 258 = 6 x 43 and 132 = 11 x 12)."""
    from paper_2006_09808_b200 import binding
    assert binding.line_factors(64) == (True, 8, 8) and binding.line_factors(256) == (True, 16, 16)
    assert binding.line_factors(512) == (True, 32, 16)          # a whole warp per row, three stages
    assert binding.line_factors(258) == (False, 6, 43) and binding.line_factors(132) == (False, 11, 12)
    for n in range(4, 1025, 2):
        tuned, n1, n2 = binding.line_factors(n)
        assert n1 * n2 == n and (tuned or n1 <= n2)
        if not tuned:   # no factor pair is more balanced
            assert all(n % f or f <= n1 for f in range(1, int(n ** 0.5) + 1))
    assert binding.line_factors(254) == (False, 2, 127)        # 2 x prime: one long dense stage
    for bad in (257, 2, 1026, 0, -4):
        with pytest.raises(binding.PdError) as e:
            binding.line_factors(bad)
        assert e.value.code == binding.ESIZE


def test_hybrid_tail_rule_host_logic(libpath):
    """pd_hybrid_tail_rule (pure host arithmetic behind PD_OPT_HYBRID_TAIL = -1): the resident clusters
    run whole waves, the tail is what is left, and it never asks the streaming side for more than it can do in that time."""
    from paper_2006_09808_b200 import binding
    rule = binding.hybrid_tail_rule
    assert rule(64, 15, 0.19) == 4        # NS: 128 slices = 64 pairs = 4 full waves of 15 + 4
    assert rule(512, 15, 0.19) == 77      # C3: 29 waves + 77 (30 waves + 62 would take one wave longer)
    assert rule(512, 15, 0.15) == 62      # a slower streaming side gets a smaller tail
    assert rule(32, 15, 0.19) == 2        # C2
    assert rule(15, 15, 0.19) == 0 and rule(30, 15, 0.19) == 0 and rule(7, 15, 0.19) == 0   # whole waves / less than one wave: no tail
    assert rule(0, 15, 0.19) == 0 and rule(10, 0, 0.19) == 0 and rule(64, 15, 0.0) == 0
    for rho in (0.08, 0.15, 0.19, 0.3):
      for ncl in (1, 7, 15, 18):
        for npairs in range(1, 400):
            t = rule(npairs, ncl, rho)
            assert 0 <= t < npairs
            assert (npairs - t) % ncl == 0 or t == 0          # the resident part is whole waves whenever a tail is split off
            w = -(-(npairs - t) // ncl)
            assert t / (rho * ncl) <= max(w, -(-npairs // ncl)) + 1e-9   # the tail never becomes the bottleneck vs no tail
            assert max(w, t / (rho * ncl)) <= -(-npairs // ncl) + 1e-9   # never slower than the pure resident schedule
