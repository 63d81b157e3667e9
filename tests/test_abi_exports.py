"""Host-only checks of the boundary: the C-ABI library builds for sm_100a, loads, and exports every symbol that
include/lqcd_b200.h declares (no compute calls: there is no GPU here)."""
import ctypes
import os
import re

from paper_2510_26313_b200 import binding, build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "lqcd_b200.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(lq_[a-z_0-9]+)\s*\(", text)) - {"lq_alloc_fn", "lq_free_fn"})


def test_library_builds_and_exports_every_declared_symbol():
    so = build.build()
    lib = ctypes.CDLL(so)
    syms = declared_symbols()
    assert len(syms) >= 15
    for s in syms:
        assert hasattr(lib, s), s
    assert sorted(binding.EXPORTS) == syms


def test_struct_layouts_match_header():
    # lq_solve_param: double,int,int,int,(pad),double,int,int,int,int ; lq_solve_info as declared
    assert ctypes.sizeof(binding.SolveParam) == 48
    assert ctypes.sizeof(binding.SolveInfo) == 4 * 3 + 4 * 16 + 4 + 8 * 16 + 8 + 8
    assert binding.LQ_MAX_RHS == 16


def test_bad_arguments_fail_without_a_gpu():
    lib = binding.load_library()
    h = ctypes.c_void_p()
    assert lib.lq_create(ctypes.byref(h), (ctypes.c_int * 4)(4, 4, 3, 8), 0, None) == binding.LQ_EINVAL
    assert lib.lq_native_bytes(None, 8, 1, 0) == 0
    assert lib.lq_last_error(None) == b"null context"


def test_product_path_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_2510_26313_b200")
    for dp, _, fs in os.walk(pkg):
        for f in fs:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dp, f)).read()
                assert "import oracle" not in src and "from oracle" not in src and "liboracle" not in src, f
