"""The C-ABI boundary without a GPU: libotoo.so loads and exports every function include/otoo.h declares
(and nothing declared is missing from the Python binding's list).  No compute call is made."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
LIB = os.path.join(ROOT, "paper_1206_1199_b200", "libotoo.so")
HDR = os.path.join(ROOT, "include", "otoo.h")


def declared_functions():
    src = open(HDR).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(otoo_[a-z0-9_]+)\s*\(", src)))


def test_header_declares_the_north_star_entry_points():
    names = declared_functions()
    for must in ("otoo_build_tree", "otoo_gravity", "otoo_sph_density", "otoo_sph_force", "otoo_gravity_delta"):
        assert must in names


def test_library_exports_every_declared_symbol():
    if not os.path.exists(LIB):
        from paper_1206_1199_b200 import build
        build.build()
    lib = ctypes.CDLL(LIB)
    for name in declared_functions():
        assert hasattr(lib, name), f"{name} is declared in include/otoo.h but not exported by libotoo.so"
    lib.otoo_version.restype = ctypes.c_int
    assert lib.otoo_version() >= 1


def test_binding_lists_every_declared_symbol():
    src = open(os.path.join(ROOT, "paper_1206_1199_b200", "binding.py")).read()
    m = re.search(r"EXPORTS = \[(.*?)\]", src, flags=re.S)
    listed = set(re.findall(r'"(otoo_[a-z0-9_]+)"', m.group(1)))
    assert listed == set(declared_functions())


def test_null_context_is_an_error_not_a_crash():
    if not os.path.exists(LIB):
        pytest.skip("library not built")
    lib = ctypes.CDLL(LIB)
    lib.otoo_gravity.argtypes = [ctypes.c_void_p, ctypes.c_float, ctypes.c_float, ctypes.c_int, ctypes.c_void_p, ctypes.c_void_p]
    assert lib.otoo_gravity(None, 0.01, 0.5, 64, None, None) == 1          # OTOO_ERR_INVALID_ARG
    lib.otoo_set_option.argtypes = [ctypes.c_void_p, ctypes.c_char_p, ctypes.c_int64]
    assert lib.otoo_set_option(None, b"task_pool", 1) == 1


def test_header_is_plain_c_and_structs_match_the_binding(tmp_path):
    """include/otoo.h compiles as C99 on its own; the ctypes mirrors in binding.py have the sizes and field offsets
    the C compiler gives otoo_stats_t / otoo_tree_info_t / otoo_cell_t (per-phase times, walk_only and error_flag are
    there: SURVEY 8(b))."""
    import subprocess
    torch = pytest.importorskip("torch")          # binding.py imports torch (CPU build is enough)
    from paper_1206_1199_b200 import binding
    fields = [n for n, _ in binding.Stats._fields_]
    for must in ("ms_build", "ms_build_total", "ms_walk_prep", "ms_walk_force", "ms_total", "walk_only", "error_flag",
                 "sum_tests", "sum_interactions"):
        assert must in fields
    prog = ['#include <stdio.h>', '#include <stddef.h>', f'#include "{HDR}"', "int main(void) {",
            '  printf("%zu %zu %zu\\n", sizeof(otoo_stats_t), sizeof(otoo_tree_info_t), sizeof(otoo_cell_t));']
    for n in fields:
        prog.append(f'  printf("{n} %zu\\n", offsetof(otoo_stats_t, {n}));')
    prog += ["  return 0;", "}"]
    src = tmp_path / "abi.c"
    src.write_text("\n".join(prog))
    exe = tmp_path / "abi"
    subprocess.run(["gcc", "-std=c99", "-Wall", "-Werror", "-o", str(exe), str(src)], check=True)
    out = subprocess.run([str(exe)], check=True, capture_output=True, text=True).stdout.split("\n")
    sizes = [int(x) for x in out[0].split()]
    assert sizes == [ctypes.sizeof(binding.Stats), ctypes.sizeof(binding.TreeInfo), binding.CELL_DTYPE.itemsize]
    for line in out[1:]:
        if line:
            n, off = line.split()
            assert getattr(binding.Stats, n).offset == int(off), n
    assert len(binding.BUILD_PHASES) <= 8
