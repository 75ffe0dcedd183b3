"""CPU-side checks of the boundary: liblya.so builds for sm_100a, loads, and exports
every symbol include/lya.h declares; without a GPU the library refuses to run."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2507_00129_b200 import build, binding
    build.build()
    return binding.load()


def _declared():
    src = open(os.path.join(ROOT, "include", "lya.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(lya_[a-z0-9_]+)\s*\(", src)))


def test_exports_every_declared_symbol(lib):
    from paper_2507_00129_b200 import binding
    names = _declared()
    assert {"lya_neighbours", "lya_xi2pcf", "lya_dmat", "lya_create", "lya_run_host"} <= set(names)
    for n in names:
        assert hasattr(lib, n), f"liblya.so does not export {n}"
    assert sorted(binding.EXPORTS) == names


def test_struct_layouts_match_header():
    from paper_2507_00129_b200 import binding
    assert C.sizeof(binding.CForests) == 12 * 8
    assert C.sizeof(binding.CBinning) == 24
    assert C.sizeof(binding.CStats) == 6 * 8 + 2 * 4


def test_no_cpu_fallback(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    h = C.c_void_p()
    st = lib.lya_create(C.byref(h), 0, None)
    assert st == 6 and not h.value                      # LYA_ERR_CUDA, no ctx
    from paper_2507_00129_b200 import binding
    with pytest.raises(RuntimeError):
        binding.Context("cuda:0")


def test_product_path_never_imports_oracle():
    """The package (binding, build, gen, csrc) must not import, include, link or dlopen oracle/."""
    pkg = os.path.join(ROOT, "paper_2507_00129_b200")
    bad = re.compile(r"(^\s*(import|from)\s+oracle\b)|(#include\s*[\"<][^\">]*oracle)|(liblya_oracle)|(lya_oracle\.c)|(orc_[a-z_]+\s*\()", re.M)
    for dirpath, _, files in os.walk(pkg):
        for fn in files:
            if fn.endswith((".py", ".cu", ".cuh", ".h")):
                assert not bad.search(open(os.path.join(dirpath, fn)).read()), fn
