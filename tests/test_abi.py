"""CPU-side checks of the boundary: the C-ABI library builds, loads and exports every symbol include/mhd.h declares;
the ctypes mirror of mhd_patch_desc has the compiled layout. No compute calls (no GPU here)."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def built_lib():
    from paper_2510_13965_b200 import build
    return build.build()


def test_library_exports_every_declared_symbol(built_lib):
    hdr = open(os.path.join(ROOT, "include", "mhd.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(mhd_[a-z0-9_]+)\s*\(", hdr))
    assert {"mhd_patch_create", "mhd_fill_ghosts", "mhd_con2prim", "mhd_rhs", "mhd_rk_stage"} <= declared
    lib = ctypes.CDLL(built_lib)
    for name in declared:
        assert hasattr(lib, name), name
    from paper_2510_13965_b200 import binding
    assert set(binding.EXPORTS) == declared


def test_desc_layout_matches(built_lib):
    from paper_2510_13965_b200 import binding
    L = binding.lib()          # raises on layout mismatch
    assert L.mhd_desc_sizeof() == ctypes.sizeof(binding.mhd_patch_desc)
    assert L.mhd_strerror(0) == b"ok" and L.mhd_strerror(-2) == b"slot not bound"


def test_argument_errors_without_gpu(built_lib):
    from paper_2510_13965_b200 import binding, synth
    L = binding.lib()
    h = ctypes.c_void_p()
    d = binding.make_desc(synth.default_params(), 8, 8, 8, 2, 0.1)      # ng < 3 is rejected before any CUDA call
    assert L.mhd_patch_create(ctypes.byref(d), ctypes.byref(h)) == -1
    assert L.mhd_patch_create(None, ctypes.byref(h)) == -1
    d = binding.make_desc(synth.default_params(), 8, 8, 8, 3, 0.1)
    d.n_species = 2                                                      # only 0 (M1 off) and 3 are built
    assert L.mhd_patch_create(ctypes.byref(d), ctypes.byref(h)) == -4


def test_product_does_not_import_oracle():
    import glob
    for f in glob.glob(os.path.join(ROOT, "paper_2510_13965_b200", "**", "*"), recursive=True):
        if f.endswith((".py", ".cu", ".cuh", ".h")):
            src = open(f).read()
            assert "import oracle" not in src and "from oracle" not in src and "orc.hpp" not in src, f
    for f in glob.glob(os.path.join(ROOT, "oracle", "*")):
        if f.endswith((".py", ".cpp", ".hpp")):
            # the seeded input generators (synth: no method arithmetic) are the one module that serves both sides
            src = open(f).read().replace("from paper_2510_13965_b200 import synth", "")
            assert "import paper_2510_13965_b200" not in src and "from paper_2510_13965_b200" not in src and "mhd.h" not in src, f
