"""CPU-side checks of the C-ABI library: it loads, exports every symbol include/mhs.h declares, and
its host logic (option defaults, argument validation, status strings) behaves.  No compute calls."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def L():
    from paper_1307_6720_b200 import binding
    return binding.lib()


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "mhs.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(mhs_[a-z0-9_]+)\s*\(", src)))


def test_header_symbols_are_exported(L):
    from paper_1307_6720_b200 import binding
    syms = declared_symbols()
    assert len(syms) >= 20
    for s in syms:
        assert hasattr(L, s), "libmhs_b200.so does not export %s" % s
    assert sorted(binding.EXPORTS) == syms                      # binding and header agree


def test_struct_sizes_match_header():
    """Compile a tiny C program against include/mhs.h and compare sizeof() with the ctypes mirrors."""
    import subprocess
    import tempfile
    from paper_1307_6720_b200 import binding as b
    with tempfile.TemporaryDirectory() as d:
        src = os.path.join(d, "s.c")
        open(src, "w").write('#include <stdio.h>\n#include "mhs.h"\nint main(){printf("%zu %zu %zu %zu %zu\\n",'
                             'sizeof(mhs_grid),sizeof(mhs_bc),sizeof(mhs_options),sizeof(mhs_solve_info),sizeof(mhs_profile));return 0;}\n')
        exe = os.path.join(d, "s")
        subprocess.run(["gcc", "-I", os.path.join(ROOT, "include"), src, "-o", exe], check=True)
        out = subprocess.run([exe], check=True, capture_output=True, text=True).stdout.split()
    want = [C.sizeof(x) for x in (b.mhs_grid, b.mhs_bc, b.mhs_options, b.mhs_solve_info, b.mhs_profile)]
    assert [int(v) for v in out] == want


def test_defaults_and_strings(L):
    from paper_1307_6720_b200 import binding as b
    o = b.mhs_options()
    L.mhs_default_options(C.byref(o))
    assert o.dtype == b.MHS_F64 and abs(o.omega - 2.0 / 3.0) < 1e-16 and (o.n_pre, o.n_post) == (2, 2)
    assert o.max_levels == 0 and o.boundary_tol == 1e-10 and o.mu0 == 0.5 and o.g == 1.0 and o.profile == 0
    assert L.mhs_status_string(0) == b"MHS_OK" and L.mhs_status_string(6) == b"MHS_ERR_NOT_CONVERGED"
    assert L.mhs_kernel_class_name(0) == b"smooth_l0"
    assert L.mhs_last_error(None) == b"null context"


def _create(L, nx, ny, nz, alpha=0.5, f=None, **ov):
    from paper_1307_6720_b200 import binding as b
    o = b.mhs_options()
    L.mhs_default_options(C.byref(o))
    for k, v in ov.items():
        setattr(o, k, v)
    g = b.mhs_grid(nx, ny, nz, 1.0, 1.0, 1.0)
    h = C.c_void_p()
    fa = (C.c_double * nz)(*f) if f is not None else None
    st = L.mhs_create(C.byref(g), alpha, fa, None, C.byref(o), C.byref(h))
    msg = L.mhs_last_error(h).decode() if h else ""
    if h:
        L.mhs_destroy(h)
    return st, msg


def test_create_validates_arguments_before_touching_the_device(L):
    from paper_1307_6720_b200 import binding as b
    assert _create(L, 34, 33, 33)[0] == b.MHS_ERR_GRID                      # odd number of intervals
    assert _create(L, 33, 33, 2)[0] == b.MHS_ERR_GRID
    assert _create(L, 33, 33, 33, f=[-1.0] * 33)[0] == b.MHS_ERR_NOT_ELLIPTIC   # xi >= 1
    assert _create(L, 33, 33, 33, omega=0.0)[0] == b.MHS_ERR_INVALID_ARG
    assert _create(L, 33, 33, 33, dtype=7)[0] == b.MHS_ERR_INVALID_ARG
    assert L.mhs_create(None, 0.0, None, None, None, None) == b.MHS_ERR_INVALID_ARG


def test_no_cpu_fallback(L):
    """Without a CUDA device the product must fail loudly (never route through a CPU path)."""
    import torch
    from paper_1307_6720_b200 import binding as b
    if torch.cuda.is_available():
        pytest.skip("CUDA device present")
    st, msg = _create(L, 33, 33, 33)
    assert st == b.MHS_ERR_CUDA and "no CPU fallback" in msg
    with pytest.raises(RuntimeError, match="no CPU fallback"):
        b.Solver(33, 33, 33)


def test_product_never_imports_the_oracle():
    """The package and bench's product path share no code with oracle/ (and vice versa)."""
    pkg = os.path.join(ROOT, "paper_1307_6720_b200")
    for dp, _, fs in os.walk(pkg):
        for f in fs:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dp, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle\b", txt, flags=re.M), f
                assert "mhs_oracle" not in txt and "orc_" not in txt, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c", ".h")):
            txt = open(os.path.join(ROOT, "oracle", f)).read()
            assert not re.search(r"^\s*(import|from)\s+paper_1307_6720_b200\b", txt, flags=re.M), f
            assert "libmhs_b200" not in txt and "binding" not in txt.replace("bindings", ""), f
