"""CPU-side checks of the boundary: the library builds, loads, and exports every symbol
include/fdham.h declares; argument validation that needs no GPU."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2310_14776_b200 import build, fdham
    build.build()
    return fdham.load_library()


def _declared_functions():
    text = open(os.path.join(ROOT, "include", "fdham.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(fd_[a-z_]+)\s*\(", text)))


def test_header_declares_the_north_star_calls():
    names = _declared_functions()
    for need in ["fd_create", "fd_apply_kinetic", "fd_apply_hamiltonian", "fd_destroy"]:
        assert need in names


def test_library_exports_every_declared_symbol(lib):
    from paper_2310_14776_b200 import fdham
    declared = _declared_functions()
    assert sorted(fdham.EXPORTED_SYMBOLS) == declared
    for name in declared:
        assert hasattr(lib, name), name


def test_strerror_strings(lib):
    from paper_2310_14776_b200 import strerror
    assert strerror(0) == "success"
    assert "alias" in strerror(-3).lower() or "overlap" in strerror(-3).lower()
    assert "unknown" in strerror(-99)


def test_create_rejects_bad_arguments_before_touching_cuda(lib):
    from paper_2310_14776_b200 import FDError, fd_create
    bad = [
        dict(shape=(0, 8, 8), h=(0.2,) * 3),
        dict(shape=(8, 8, 8), h=(0.2, -1.0, 0.2)),
        dict(shape=(8, 8, 8), h=(0.2, float("nan"), 0.2)),
        dict(shape=(8, 8, 8), h=(0.2,) * 3, nn=0),
        dict(shape=(8, 8, 8), h=(0.2,) * 3, nn=7),
        dict(shape=(8, 8, 8), h=(0.2,) * 3, bc=(1, 2, 1)),
        dict(shape=(2, 8, 8), h=(0.2,) * 3, bc=(1, 1, 1)),            # periodic axis shorter than nn
        dict(shape=(8, 8, 8), h=(0.2,) * 3, k=(0.25, 0, 0)),          # real dtype with k != 0
        dict(shape=(8, 8, 8), h=(0.2,) * 3, bc=(0, 1, 1), k=(0.25, 0, 0), dtype=1),  # k on zero axis
        dict(shape=(8, 8, 8), h=(0.2,) * 3, dtype=5),
    ]
    for kw in bad:
        with pytest.raises(FDError) as ei:
            fd_create(**kw)
        assert ei.value.status == -1, kw


def test_no_cpu_fallback_without_device(lib):
    """On a box without a GPU a valid fd_create must fail loudly with FD_ERR_CUDA."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    from paper_2310_14776_b200 import FDError, fd_create
    with pytest.raises(FDError) as ei:
        fd_create((8, 8, 8), (0.2,) * 3)
    assert ei.value.status == -4


def test_null_plan_rejected(lib):
    assert lib.fd_apply_kinetic(None, None, None, 1, None) == -1
    assert lib.fd_apply_hamiltonian(None, None, None, None, 1, None) == -1
    assert lib.fd_destroy(None) == 0
    assert lib.fd_plan_get_kernel(None) == -1


def test_product_path_does_not_import_oracle():
    """The package and bench product path must not route through oracle/."""
    pkg = os.path.join(ROOT, "paper_2310_14776_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".h", ".cpp")):
                src = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in src.replace("no CPU", ""), f


def test_c_abi_from_plain_c(lib, tmp_path):
    """include/fdham.h compiles as C99 (-Wall -Wextra -pedantic -Werror) and libfdham.so links and
    runs from a C program with no C++ / torch dependency."""
    import subprocess
    from paper_2310_14776_b200 import fdham
    exe = tmp_path / "c_abi_check"
    libdir = os.path.dirname(fdham.LIB_PATH)
    cmd = ["gcc", "-std=c99", "-Wall", "-Wextra", "-pedantic", "-Werror", "-I", os.path.join(ROOT, "include"),
           os.path.join(ROOT, "tests", "c_abi_check.c"), "-o", str(exe), "-L", libdir, "-lfdham",
           "-Wl,-rpath," + libdir]
    res = subprocess.run(cmd, capture_output=True, text=True)
    assert res.returncode == 0, res.stderr
    run = subprocess.run([str(exe)], capture_output=True, text=True, timeout=120)
    assert run.returncode == 0, (run.returncode, run.stdout, run.stderr)
    assert "c_abi_check" in run.stdout
