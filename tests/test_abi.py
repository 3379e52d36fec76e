"""CPU-side checks of the C-ABI library (-m "not gpu"): it builds for sm_100a, loads without a GPU, exports every
symbol include/lqcd_b200.h declares, and its pure-host logic (sizes, knob validation) behaves.  No compute calls."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "lqcd_b200.h")


def declared_symbols():
    text = open(HEADER).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(lqcd_[a-z0-9_]+)\s*\(", text)))


@pytest.fixture(scope="module")
def lib():
    from paper_2111_05012_b200 import _lib
    return _lib.load()


def test_header_declares_the_survey_entry_points():
    syms = declared_symbols()
    for base in ("wilson_clover_mult", "coarse_mult", "restrict", "prolong", "pack_spinor", "unpack_spinor",
                 "pack_gauge", "pack_clover", "pack_nullvec"):
        for p in ("f32", "f64"):
            assert f"lqcd_{base}_{p}" in syms
    assert "lqcd_last_error" in syms and "lqcd_version" in syms


def test_library_exports_every_declared_symbol(lib):
    from paper_2111_05012_b200 import _lib
    syms = declared_symbols()
    assert len(syms) >= 36
    for s in syms:
        assert hasattr(lib, s), f"{s} declared in the header but not exported"
    assert set(_lib.SIGNATURES) == set(syms), "python binding table and header disagree"


def test_library_is_sm100a_only():
    from paper_2111_05012_b200 import _lib
    import subprocess, shutil
    cuobjdump = shutil.which("cuobjdump") or "/usr/local/cuda/bin/cuobjdump"
    if not os.path.exists(cuobjdump):
        pytest.skip("cuobjdump not available")
    out = subprocess.run([cuobjdump, "-lelf", _lib.lib_path()], capture_output=True, text=True).stdout
    archs = set(re.findall(r"sm_\d+a?", out))
    assert archs == {"sm_100a"}, archs


def test_host_logic_sizes_and_knobs(lib):
    i4 = C.c_int * 4
    dims, block = i4(48, 48, 48, 96), i4(4, 4, 4, 4)
    V = 48 ** 3 * 96
    assert lib.lqcd_version() >= 100
    assert lib.lqcd_native_spinor_reals(dims) == V * 24
    assert lib.lqcd_native_gauge_reals(dims, 0) == V * 72
    assert lib.lqcd_native_gauge_reals(dims, 2) == V * 48
    assert lib.lqcd_native_clover_reals(dims) == V * 72
    assert lib.lqcd_native_nullvecs_reals(dims, block, 32) == V * 24 * 32
    cd = i4(12, 12, 12, 24)
    assert lib.lqcd_native_coarse_vec_reals(cd, 32) == 12 ** 3 * 24 * 128
    assert lib.lqcd_native_coarse_mat_reals(cd, 32) == 12 ** 3 * 24 * 9 * 64 * 64 * 2
    # ragged volume is padded to whole chunks of 32 sites
    assert lib.lqcd_native_spinor_reals(i4(3, 3, 3, 3)) == 96 * 24
    # invalid geometry -> 0
    assert lib.lqcd_native_spinor_reals(i4(4, 4, 0, 4)) == 0
    assert lib.lqcd_native_nullvecs_reals(dims, i4(5, 4, 4, 4), 32) == 0
    # coarse extent 1 is fine for the aggregate-local operations (a rank of a sharded lattice may be one aggregate
    # thick); only the periodic 9-point coarse stencil needs extents >= 2 (Q8)
    assert lib.lqcd_native_nullvecs_reals(i4(4, 4, 4, 4), block, 4) == 256 * 24 * 4
    # knobs
    assert lib.lqcd_set_fine_tile(i4(8, 4, 4, 1)) == 0
    assert lib.lqcd_set_fine_tile(i4(8, 8, 8, 8)) == -1
    assert b"threads per CTA" in lib.lqcd_last_error()
    assert lib.lqcd_set_fine_tile(None) == 0
    assert lib.lqcd_set_knob(b"no_such_knob", 1) == -1
    assert lib.lqcd_set_knob(b"fine_tslab", 0) == 0
    assert lib.lqcd_host_workspace_bytes(i4(8, 8, 8, 8), i4(4, 4, 4, 4), 16) >= 3 * 4096 * 96 + 2 * 16 * 32 * 8


def test_product_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_2111_05012_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle\b", text, flags=re.M), f
                assert "lqcd_oracle" not in text, f
