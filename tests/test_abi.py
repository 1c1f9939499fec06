"""CPU-side checks of the C-ABI boundary: the library builds, loads, exports every symbol the header declares,
and fails loudly (no fallback) without a GPU."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_1507_08549_b200 import build, binding
    build.build()
    return binding.load()


def header_symbols():
    """Every function any include/*.h declares."""
    out = set()
    for fn in sorted(os.listdir(os.path.join(ROOT, "include"))):
        if fn.endswith(".h"):
            src = open(os.path.join(ROOT, "include", fn)).read()
            src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
            out |= set(re.findall(r"\b(sn_[a-z0-9_]+)\s*\(", src))
    return sorted(out)


def test_header_and_binding_agree():
    from paper_1507_08549_b200 import binding
    exports = list(binding.EXPORTS) + [x for name in dir(binding) if name.startswith("EXPORTS_")
                                       for x in getattr(binding, name)]
    assert header_symbols() == sorted(exports)


def test_library_exports_every_declared_symbol(lib):
    for name in header_symbols():
        assert hasattr(lib, name), name


def test_result_struct_is_16_bytes():
    from paper_1507_08549_b200 import sn_poisson_result
    assert C.sizeof(sn_poisson_result) == 16


def test_create_rejects_bad_arguments_or_missing_gpu(lib):
    from paper_1507_08549_b200 import binding
    import torch
    bad = [(1, 8, .1, .1, 1, 4), (8, 8, -1., .1, 1, 4), (8, 8, .1, float("nan"), 1, 4), (8, 8, .1, .1, 2, 4),
           (8, 8, .1, .1, 1, -1), (8, 8, .1, .1, 1, 65)]
    for a in bad:
        assert not lib.sn_poisson_create(*a)
        assert binding.sn_poisson_last_error() != ""
    if not torch.cuda.is_available():
        # no device: the product must refuse, not fall back to a CPU path
        assert not lib.sn_poisson_create(8, 8, .1, .1, 1, 4)
        with pytest.raises(binding.SnPoissonError):
            binding.sn_poisson_create(8, 8, .1, .1, 1, 4)


def test_null_handle_is_an_error_not_a_crash(lib):
    r = lib.sn_poisson_solve(None, None, None, 1e-10, 10, None)
    assert r.status == -1 and r.sweeps == 0
    assert lib.sn_poisson_set_omega(None, 1.5) == -1
    lib.sn_poisson_destroy(None)


def test_product_does_not_import_the_oracle():
    """Neither side imports the other: no import / include / dlopen of anything under oracle/ in the package."""
    pkg = os.path.join(ROOT, "paper_1507_08549_b200")
    pat = re.compile(r"(import\s+oracle|from\s+oracle|oracle/|sn_oracle|sno_)")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".cpp")):
                assert not pat.search(open(os.path.join(dirpath, f)).read()), (dirpath, f)
    orc = open(os.path.join(ROOT, "oracle", "__init__.py")).read()
    assert not re.search(r"^\s*(import|from)\s+paper_1507_08549_b200", orc, flags=re.M)
    cpp = open(os.path.join(ROOT, "oracle", "sn_oracle.cpp")).read()
    assert not re.search(r'#include\s+"[^"]*(csrc|sn_poisson|common\.cuh)', cpp)
