"""CPU-only checks of the boundary: the C-ABI library loads without a GPU, exports every symbol
include/synim.h declares, and its pure-host helper agrees with the oracle's independent
composition.  No compute entry point is exercised here."""
import ctypes
import math
import os
import re

import numpy as np
import pytest

from oracle import oracle as O
from paper_2606_07759_b200 import build, synim
from paper_2606_07759_b200 import workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    build.build_library()
    return synim.lib()


def test_library_exports_every_declared_symbol(lib):
    header = open(os.path.join(ROOT, "include", "synim.h")).read()
    header = re.sub(r"/\*.*?\*/", "", header, flags=re.S)
    declared = set(re.findall(r"\b(synim_[a-z_0-9]+)\s*\(", header))
    assert declared == set(synim.EXPORTS)
    for name in declared:
        assert getattr(lib, name) is not None
    assert synim.version() == 3


def test_compose_affine_matches_the_oracles_independent_composition(lib):
    rng = np.random.default_rng(21)
    for _ in range(20):
        phys = W.physical(shift_x=rng.uniform(-2, 2), shift_y=rng.uniform(-2, 2), rot_deg=rng.uniform(-180, 180),
                          mag_x=rng.uniform(0.8, 1.2), mag_y=rng.uniform(0.8, 1.2),
                          dm_shift_x=rng.uniform(-2, 2), dm_shift_y=rng.uniform(-2, 2),
                          dm_rot_deg=rng.uniform(-10, 10), dm_mag=rng.uniform(0.9, 1.1),
                          dm_height_m=rng.uniform(0, 20000), gs_range_m=rng.choice([math.inf, 90000.0]),
                          gs_theta_arcsec=rng.uniform(0, 80), gs_azimuth_deg=rng.uniform(0, 360),
                          src_pixel_pitch_m=rng.uniform(0.05, 0.1), wfs_pitch_src_px=rng.uniform(0.98, 1.02))
        assert np.allclose(synim.compose_affine(phys), O.compose_affine(phys), rtol=0, atol=1e-9)
    assert np.array_equal(synim.compose_affine(W.physical()), [1, 0, 0, 0, 1, 0])
    for cfg in (1, 2, 3, 4):
        wl = W.make_config(cfg, max_modes=1)
        for w in wl.wfs:
            assert np.allclose(synim.compose_affine(w.phys), O.compose_affine(w.phys), rtol=0, atol=1e-10)


def test_argument_errors_are_reported_not_thrown(lib):
    bad = W.physical(mag_x=0.0)
    with pytest.raises(synim.SynimError) as e:
        synim.compose_affine(bad)
    assert e.value.status == synim.ERR_INVALID_ARG and "magnification" in synim.last_error()
    # NULL-safe calls that never reach CUDA
    lib.synim_destroy(None)
    assert lib.synim_num_rows(None) == -1 and lib.synim_num_valid(None, 0) == -1
    assert lib.synim_create_geometry(8, 8, 1, None, None, None) == synim.ERR_INVALID_ARG
    h = ctypes.c_void_p()
    g = (synim.WfsGrid * 1)()
    assert lib.synim_create_geometry(8, 8, 0, g, None, ctypes.byref(h)) == synim.ERR_INVALID_ARG
    assert lib.synim_create_geometry(8, 10, 1, g, None, ctypes.byref(h)) == synim.ERR_ALIGNMENT
    assert lib.synim_interaction_matrix(None, None, 1, None, None, 0, 0, None, 0, None, 1, None) == synim.ERR_INVALID_ARG
    w, hh = ctypes.c_int32(), ctypes.c_int32()
    assert lib.synim_bbox_extent(None, 0, ctypes.byref(w), ctypes.byref(hh), None) == synim.OK


def test_product_code_never_touches_the_oracle():
    """The oracle is test infrastructure: nothing under the package may import or load it."""
    pkg = os.path.join(ROOT, "paper_2606_07759_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".h", ".cuh", ".cpp")):
                text = open(os.path.join(dirpath, f)).read()
                assert "liboracle" not in text and "import oracle" not in text and "from oracle" not in text, f
    otext = open(os.path.join(ROOT, "oracle", "oracle.py")).read() + open(os.path.join(ROOT, "oracle", "synim_oracle.c")).read()
    assert "libsynim" not in otext and "paper_2606_07759_b200" not in otext.replace("paper_2606_07759_b200/csrc", "")


def test_header_is_plain_c_and_links_from_c(tmp_path):
    """include/synim.h is the boundary: it compiles as strict C11 and as C++17, and a C program that includes it links
    against the library and reaches the entry points that need no GPU (version, argument errors, NULL-safe destroy)."""
    import shutil
    import subprocess
    hdr = os.path.join(ROOT, "include", "synim.h")
    subprocess.check_call(["gcc", "-std=c11", "-Wall", "-Wextra", "-pedantic", "-Werror", "-fsyntax-only", "-x", "c", hdr])
    subprocess.check_call(["g++", "-std=c++17", "-Wall", "-Werror", "-fsyntax-only", "-x", "c++", hdr])
    src = tmp_path / "use.c"
    src.write_text(
        '#include "synim.h"\n#include <stdio.h>\n#include <string.h>\n'
        "int main(void) {\n"
        "  synim_wfs_affine a; synim_wfs_physical p; memset(&p, 0, sizeof p);\n"
        "  if (synim_version() != SYNIM_VERSION_MAJOR * 1000 + SYNIM_VERSION_MINOR) return 1;\n"
        "  if (synim_compose_affine(&p, &a) != SYNIM_ERR_INVALID_ARG) return 2;   /* zero magnification */\n"
        "  if (strlen(synim_last_error()) == 0) return 3;\n"
        "  if (synim_num_rows(NULL) != -1) return 4;\n"
        "  synim_destroy(NULL);\n"
        "  if (synim_interaction_matrix(NULL, NULL, 0, NULL, NULL, 0, 0, NULL, SYNIM_SLOPES_ND, NULL, 0, NULL) != SYNIM_ERR_INVALID_ARG) return 5;\n"
        '  printf("ok %d\\n", (int)synim_version());\n  return 0;\n}\n')
    exe = tmp_path / "use"
    shutil.copy(synim.LIB_PATH, tmp_path / "libsynim.so")
    subprocess.check_call(["gcc", "-std=c11", "-Wall", "-Werror", "-I", os.path.join(ROOT, "include"), str(src), "-o", str(exe),
                           "-L", str(tmp_path), "-lsynim", "-Wl,-rpath," + str(tmp_path)])
    out = subprocess.run([str(exe)], capture_output=True, text=True)
    assert out.returncode == 0, (out.returncode, out.stdout, out.stderr)
    assert out.stdout.startswith("ok ")
