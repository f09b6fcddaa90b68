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


def test_header_compiles_as_c99_and_layouts_match_field_by_field(built_lib, tmp_path):
    """include/mhd.h is a C header: a C99 translation unit includes it, prints offsetof / sizeof of every field of mhd_patch_desc,
    mhd_tableau and mhd_status as the C compiler lays them out, and drives the error paths through the linked library; the ctypes
    mirrors in binding.py must agree field by field (a size check alone would not see two swapped doubles)."""
    import subprocess
    from paper_2510_13965_b200 import binding
    structs = {"mhd_patch_desc": binding.mhd_patch_desc, "mhd_tableau": binding.mhd_tableau, "mhd_status": binding.mhd_status}
    lines = []
    for sname, cls in structs.items():
        for fname, _ in cls._fields_:
            lines.append('  printf("%s.%s %%zu %%zu\\n", offsetof(%s, %s), sizeof(((%s*)0)->%s));' % (sname, fname, sname, fname, sname, fname))
        lines.append('  printf("%s.sizeof %%zu 0\\n", sizeof(%s));' % (sname, sname))
    src = tmp_path / "abi.c"
    src.write_text('#include <stdio.h>\n#include <stddef.h>\n#include "mhd.h"\nint main(void) {\n' + "\n".join(lines) + '''
  mhd_patch *p = NULL;
  mhd_patch_desc d = {0};
  int bc[6] = {0, 0, 0, 0, 0, 0};
  printf("rc.null_desc %d 0\\n", mhd_patch_create(NULL, &p));
  d.nx = d.ny = d.nz = 8; d.ng = 2; d.dx = d.dy = d.dz = 0.1;
  printf("rc.ng2 %d 0\\n", mhd_patch_create(&d, &p));
  d.ng = 3; d.recon_kind = 7;
  printf("rc.recon %d 0\\n", mhd_patch_create(&d, &p));
  d.recon_kind = 0; d.les_C_M = 8.0;
  printf("rc.les_ng3 %d 0\\n", mhd_patch_create(&d, &p));
  printf("rc.fill_null %d 0\\n", mhd_fill_ghosts(NULL, MHD_SLOT_U, bc, NULL));
  printf("rc.dense_scheme %d 0\\n", mhd_dense_weights(5, 0.5, 0, (double[4]){0}));
  printf("str.unbound %s 0\\n", mhd_strerror(MHD_E_UNBOUND)[0] == 's' ? "1" : "0");
  printf("enum.nslots %d 0\\n", (int)MHD_NSLOTS);
  return 0;
}
''')
    exe = tmp_path / "abi"
    libdir = os.path.dirname(built_lib)
    subprocess.run(["gcc", "-std=c99", "-Wall", "-Werror", "-pedantic", "-I", os.path.join(ROOT, "include"), str(src), "-o", str(exe),
                    "-L", libdir, "-lmhd_b200", "-Wl,-rpath," + libdir], check=True)
    out = subprocess.run([str(exe)], check=True, capture_output=True, text=True).stdout
    got = {ln.split()[0]: ln.split()[1:] for ln in out.strip().splitlines()}
    for sname, cls in structs.items():
        for fname, _ in cls._fields_:
            f = getattr(cls, fname)
            assert [int(x) for x in got["%s.%s" % (sname, fname)]] == [f.offset, f.size], (sname, fname)
        assert int(got[sname + ".sizeof"][0]) == ctypes.sizeof(cls)
    assert got["rc.null_desc"][0] == "-1" and got["rc.ng2"][0] == "-1" and got["rc.recon"][0] == "-1"
    assert got["rc.les_ng3"][0] == "-4" and got["rc.fill_null"][0] == "-1" and got["rc.dense_scheme"][0] == "-1"
    assert got["str.unbound"][0] == "1"
    assert int(got["enum.nslots"][0]) == binding.SLOT_LESWORK + 1
