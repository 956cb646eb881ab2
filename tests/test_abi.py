"""Boundary checks that need no GPU: librketd.so builds, loads, and exports exactly what include/rketd.h
declares; the Python binding carries the same names; the product path never reaches the oracle; compute
entry points fail loudly (no CPU fallback) when there is no CUDA device."""
import ctypes
import os
import re
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "rketd.h")


def declared_functions():
    src = open(HEADER).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(rketd_[a-z_]+)\s*\(", src)))


@pytest.fixture(scope="module")
def lib_path():
    from paper_1709_00821_b200 import build
    return build.build_library()


def test_header_declares_the_north_star_entry_points():
    names = declared_functions()
    for n in ("rketd_create", "rketd_set_media", "rketd_set_source", "rketd_set_probes", "rketd_run",
              "rketd_read_probes"):
        assert n in names


def test_library_exports_every_declared_symbol(lib_path):
    dll = ctypes.CDLL(lib_path)
    for n in declared_functions():
        assert hasattr(dll, n), n
    out = subprocess.run(["nm", "-D", "--defined-only", lib_path], capture_output=True, text=True, check=True).stdout
    exported = sorted(set(re.findall(r" T (rketd_[a-z_]+)$", out, flags=re.M)))
    assert exported == declared_functions()          # nothing undeclared leaks out under the rketd_ prefix


def test_binding_has_the_same_names(lib_path):
    from paper_1709_00821_b200 import rketd
    assert sorted(rketd.EXPORTS) == declared_functions()
    for n in rketd.EXPORTS:
        assert callable(getattr(rketd, n)), n


def test_header_compiles_as_plain_c(tmp_path):
    c = tmp_path / "t.c"
    c.write_text('#include "rketd.h"\nint main(void) { rketd_sim *s = 0; (void)s; return RKETD_OK; }\n')
    subprocess.run(["gcc", "-std=c99", "-Wall", "-Werror", "-I", os.path.join(ROOT, "include"), "-c", str(c),
                    "-o", str(tmp_path / "t.o")], check=True)


def test_sass_has_tma_and_fp64_fma(lib_path):
    """The temporal-blocking kernel stages tiles with TMA (UTMALDG / UTMASTG in SASS) and computes with DFMA."""
    sass = subprocess.run(["cuobjdump", "-sass", lib_path], capture_output=True, text=True, check=True).stdout
    assert "sm_100a" in sass or "SM100" in sass.upper()
    assert "UTMALDG" in sass and "UTMASTG" in sass and "DFMA" in sass


def test_product_path_is_independent_of_the_oracle():
    pkg = os.path.join(ROOT, "paper_1709_00821_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle\b", txt, flags=re.M), f
                assert "liboracle" not in txt and "rketd_oracle" not in txt, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".cpp")):
            txt = open(os.path.join(ROOT, "oracle", f)).read()
            assert "import paper_1709_00821_b200" not in txt and "from paper_1709_00821_b200" not in txt, f
            assert "librketd.so" not in txt and "rketd.h" not in txt and "csrc" not in txt, f


def test_no_cpu_fallback_without_a_device(lib_path):
    """On a box without a GPU rketd_create must fail with RKETD_ECUDA and say why."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    code = ("import sys; sys.path.insert(0, %r)\n"
            "from paper_1709_00821_b200 import rketd\n"
            "try:\n"
            "    rketd.Sim(100, 1, 75e-6, 1.25e-13)\n"
            "except rketd.RketdError as e:\n"
            "    assert e.code == rketd.ECUDA, e.code\n"
            "    assert 'no CPU fallback' in str(e)\n"
            "    print('OK')\n" % ROOT)
    out = subprocess.run([sys.executable, "-c", code], capture_output=True, text=True)
    assert out.stdout.strip() == "OK", out.stdout + out.stderr


# ---- the 2-D TMz entry points (include/rketd2d.h) ---------------------------------------------
HEADER2D = os.path.join(ROOT, "include", "rketd2d.h")


def test_2d_streaming_kernel_loads_rows_by_tma(lib_path):
    """k2_2d takes its rows as 2-D TMA boxes: every instantiation of it has UTMALDG in its SASS (and no LDGSTS row copies)."""
    sass = subprocess.run(["cuobjdump", "-sass", lib_path], capture_output=True, text=True, check=True).stdout
    funcs = re.split(r"\n\s*Function : ", sass)
    k2 = [f for f in funcs if "k2_2d" in f.split("\n", 1)[0]]
    assert len(k2) >= 10
    for f in k2:
        assert "UTMALDG" in f and "LDGSTS" not in f, f.split("\n", 1)[0]


def declared_functions_2d():
    src = re.sub(r"/\*.*?\*/", "", open(HEADER2D).read(), flags=re.S)
    return sorted(set(re.findall(r"\b(rketd2d_[a-z_]+)\s*\(", src)))


def test_library_exports_every_declared_2d_symbol(lib_path):
    dll = ctypes.CDLL(lib_path)
    names = declared_functions_2d()
    assert "rketd2d_create" in names and "rketd2d_run" in names and "rketd2d_read_probes" in names
    for n in names:
        assert hasattr(dll, n), n
    out = subprocess.run(["nm", "-D", "--defined-only", lib_path], capture_output=True, text=True, check=True).stdout
    assert sorted(set(re.findall(r" T (rketd2d_[a-z_]+)$", out, flags=re.M))) == names


def test_2d_binding_has_the_same_names(lib_path):
    from paper_1709_00821_b200 import rketd2d
    assert sorted(rketd2d.EXPORTS) == declared_functions_2d()
    for n in rketd2d.EXPORTS:
        assert callable(getattr(rketd2d, n)), n


def test_2d_header_compiles_as_plain_c(tmp_path):
    c = tmp_path / "t.c"
    c.write_text('#include "rketd2d.h"\nint main(void) { rketd2d_sim *s = 0; (void)s; return RKETD2D_BC_MUR; }\n')
    subprocess.run(["gcc", "-std=c99", "-Wall", "-Werror", "-I", os.path.join(ROOT, "include"), "-c", str(c),
                    "-o", str(tmp_path / "t.o")], check=True)


def test_2d_has_no_cpu_fallback_without_a_device(lib_path):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    code = ("import sys; sys.path.insert(0, %r)\n"
            "from paper_1709_00821_b200 import rketd2d, rketd\n"
            "try:\n"
            "    rketd2d.Sim2D(100, 100, 75e-6, 75e-6, 1.25e-13)\n"
            "except rketd.RketdError as e:\n"
            "    assert e.code == rketd.ECUDA, e.code\n"
            "    assert 'no CPU fallback' in str(e)\n"
            "    print('OK')\n" % ROOT)
    out = subprocess.run([sys.executable, "-c", code], capture_output=True, text=True)
    assert out.stdout.strip() == "OK", out.stdout + out.stderr
