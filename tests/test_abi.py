"""CPU-side checks of the boundary: the C-ABI library builds for sm_100a, loads, and exports every symbol that
include/splotch.h declares; the Python binding's struct layouts match the header.  No compute calls."""
import ctypes as C
import os
import re
import subprocess

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "splotch.h")


def declared_functions():
    src = open(HEADER).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(splotch_[a-z_]+)\s*\(", src)))


@pytest.fixture(scope="module")
def lib_path():
    from paper_1309_1114_b200 import build
    return build.build_library()


def test_header_declares_the_five_north_star_entry_points():
    names = declared_functions()
    for f in ("splotch_create", "splotch_set_camera", "splotch_set_colormap", "splotch_render", "splotch_destroy"):
        assert f in names


def test_library_exports_every_declared_symbol(lib_path):
    from paper_1309_1114_b200 import binding
    lib = C.CDLL(lib_path)
    for f in declared_functions():
        assert hasattr(lib, f), f
    assert sorted(binding.EXPORTS) == declared_functions()
    assert b"sm_100a" in C.c_char_p(C.cast(lib.splotch_version, C.CFUNCTYPE(C.c_char_p))()).value


def test_library_contains_sm100a_code_only(lib_path):
    out = subprocess.run(["cuobjdump", "--list-elf", lib_path], capture_output=True, text=True).stdout
    archs = set(re.findall(r"sm_\d+a?", out))
    assert archs == {"sm_100a"}, archs


def test_binding_struct_layouts_match_the_header(lib_path, tmp_path):
    """Compile a tiny C program against the header and compare sizeof/offsetof with the ctypes mirrors."""
    from paper_1309_1114_b200 import binding as b
    prog = tmp_path / "layout.c"
    prog.write_text(
        '#include <stdio.h>\n#include <stddef.h>\n#include "splotch.h"\nint main(void){\n'
        'printf("%zu %zu %zu %zu\\n", sizeof(splotch_particles), sizeof(splotch_species_params), sizeof(splotch_params), sizeof(splotch_stats));\n'
        'printf("%zu %zu %zu\\n", offsetof(splotch_particles, species_offsets), offsetof(splotch_params, species), offsetof(splotch_stats, stage_ms));\n'
        'return 0;}\n')
    exe = tmp_path / "layout"
    subprocess.run(["gcc", "-I", os.path.join(ROOT, "include"), "-o", str(exe), str(prog)], check=True)
    a, c = subprocess.run([str(exe)], capture_output=True, text=True, check=True).stdout.split("\n")[:2]
    assert [int(v) for v in a.split()] == [C.sizeof(b.SplotchParticles), C.sizeof(b.SplotchSpeciesParams),
                                           C.sizeof(b.SplotchParams), C.sizeof(b.SplotchStats)]
    assert [int(v) for v in c.split()] == [b.SplotchParticles.species_offsets.offset, b.SplotchParams.species.offset,
                                           b.SplotchStats.stage_ms.offset]


def test_compute_entry_points_fail_loudly_without_a_gpu(lib_path):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    from paper_1309_1114_b200 import binding as b
    with pytest.raises(b.SplotchError) as e:
        b.splotch_create(0, 64, 64, 1000)
    assert e.value.code == b.SPLOTCH_ECUDA
