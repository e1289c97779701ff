"""CPU checks of the boundary: libqs.so builds, loads, and exports every symbol include/qs.h declares."""
import ctypes
import os
import re

import paper_2403_07666_b200 as pkg
from paper_2403_07666_b200 import binding

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def header_symbols():
    src = open(os.path.join(ROOT, "include", "qs.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(qs_[a-z0-9_]+)\s*\(", src)))


def test_library_builds_loads_and_exports_every_declared_symbol():
    lib = pkg.load_library()
    names = header_symbols()
    assert len(names) >= 18 and {"qs_init", "qs_step", "qs_read"} <= set(names)
    for name in names:
        assert hasattr(lib, name), name
    assert sorted(n for n, _, _ in binding.SYMBOLS) == names


def test_struct_layouts_match_the_header(tmp_path):
    # compile include/qs.h as plain C with gcc and compare sizeof / offsetof with the ctypes mirrors
    import subprocess
    src = tmp_path / "sz.c"
    src.write_text('''#include <stdio.h>
#include <stddef.h>
#include "qs.h"
int main(void) {
  printf("%zu %zu %zu %zu %zu %zu %zu\\n", sizeof(qs_geometry), sizeof(qs_material), sizeof(qs_stats_t),
         offsetof(qs_geometry, softening), offsetof(qs_geometry, flags), offsetof(qs_material, cg_maxit),
         offsetof(qs_stats_t, launches));
  return 0;
}
''')
    exe = tmp_path / "sz"
    subprocess.run(["gcc", "-std=c99", "-I", os.path.join(ROOT, "include"), str(src), "-o", str(exe)], check=True)
    got = [int(v) for v in subprocess.run([str(exe)], capture_output=True, text=True, check=True).stdout.split()]
    G, M, S = binding.QsGeometry, binding.QsMaterial, binding.QsStats
    assert got == [ctypes.sizeof(G), ctypes.sizeof(M), ctypes.sizeof(S), G.softening.offset, G.flags.offset,
                   M.cg_maxit.offset, S.launches.offset]


def test_argument_errors_need_no_gpu():
    lib = pkg.load_library()
    g = binding.QsGeometry()
    assert lib.qs_workspace_bytes(ctypes.byref(g)) == 0
    assert b"geometry" in lib.qs_last_error()
    assert lib.qs_step(None, 1e-4, 0.0) == -1
    assert lib.qs_read(None, None, None, None, None) == -1


def test_product_does_not_import_the_oracle():
    pk = os.path.join(ROOT, "paper_2403_07666_b200")
    for dirpath, _, files in os.walk(pk):
        for f in files:
            text = open(os.path.join(dirpath, f), errors="ignore").read() if f.endswith((".py", ".cu", ".cuh", ".h")) else ""
            assert not re.search(r"^\s*(from|import)\s+oracle", text, flags=re.M), f
            assert not re.search(r"#include[^\n]*oracle", text), f
            assert "qs_oracle" not in text, f
    orc = open(os.path.join(ROOT, "oracle", "qs_oracle.py")).read()
    assert not re.search(r"^\s*(from|import)\s+paper_2403_07666_b200", orc, flags=re.M)
    assert "libqs" not in orc and "ctypes" not in orc
