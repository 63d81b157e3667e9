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


def test_struct_layouts_match_header(tmp_path):
    """sizeof / offsetof of every struct of the header, as a C compiler sees them, against the ctypes mirrors."""
    import subprocess
    structs = {"lq_solve_param": (binding.SolveParam, ["tol", "max_outer", "max_inner", "inner_prec", "delta", "check_every", "use_graph",
                                                       "keep_direction", "algorithm", "use_x0"]),
               "lq_solve_info": (binding.SolveInfo, ["nrhs", "outer_cycles", "inner_iters", "iters", "true_rel_residual", "seconds", "dslash_applies",
                                                     "model_bytes", "model_flops"]),
               "lq_eig_param": (binding.EigParam, ["n_ev", "m", "cheb_degree", "max_restarts", "cheb_a", "cheb_b", "tol", "seed"]),
               "lq_mg_param": (binding.MgParam, ["block", "n_vec", "nu_pre", "nu_post", "smoother", "coarse_iters", "restart", "setup_tol", "seed", "refine"]),
               "lq_mg_info": (binding.MgInfo, ["coarse_dims", "coarse_dof", "probes", "seconds_vectors", "seconds_prolongator", "seconds_coarse_op", "bytes"]),
               "lq_mg_solve_info": (binding.MgSolveInfo, ["iters", "outer_cycles", "true_rel_residual", "seconds", "m_applies"]),
               "lq_eig_info": (binding.EigInfo, ["restarts", "converged", "lap_applies", "max_ritz_residual", "max_true_residual", "seconds", "seconds_ritz", "seconds_ortho"])}
    lines = ['#include <stdio.h>', '#include <stddef.h>', '#include "lqcd_b200.h"', 'int main(void) {']
    for name, (_, fields) in structs.items():
        lines.append('printf("%s %%zu\\n", sizeof(%s));' % (name, name))
        for f in fields:
            lines.append('printf("%s.%s %%zu\\n", offsetof(%s, %s));' % (name, f, name, f))
    lines.append('printf("LQ_MAX_RHS %d\\n", LQ_MAX_RHS); return 0; }')
    src = tmp_path / "layout.c"
    src.write_text("\n".join(lines))
    exe = tmp_path / "layout"
    subprocess.run(["gcc", "-I", os.path.join(ROOT, "include"), "-o", str(exe), str(src)], check=True)
    got = dict(l.split() for l in subprocess.run([str(exe)], check=True, capture_output=True, text=True).stdout.splitlines())
    assert int(got["LQ_MAX_RHS"]) == binding.LQ_MAX_RHS == 32
    for name, (cls, fields) in structs.items():
        assert ctypes.sizeof(cls) == int(got[name]), name
        assert [f for f, _ in cls._fields_] == fields, name
        for f in fields:
            assert getattr(cls, f).offset == int(got[name + "." + f]), (name, f)


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
