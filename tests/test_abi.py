"""The C-ABI boundary: the shared library loads, exports every symbol include/bioem.h declares, the Python
binding carries the same names, and the calls that need no device behave as documented.  No compute calls here."""
import ctypes
import re
import subprocess
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parent.parent
HEADER = ROOT / "include" / "bioem.h"


def _declared():
    text = re.sub(r"/\*.*?\*/", "", HEADER.read_text(), flags=re.S)
    return sorted(set(re.findall(r"\b(bioem_[a-z0-9_]+)\s*\(", text)))


@pytest.fixture(scope="module")
def library():
    import paper_1609_06634_b200 as B
    from paper_1609_06634_b200 import build
    build.build()
    return B.lib()


def test_header_is_plain_c():
    """extern "C", plain pointers and sizes, no torch / C++ types in the signatures: the header compiles as C."""
    src = '#include "bioem.h"\nint main(void) { return BIOEM_OK; }\n'
    r = subprocess.run(["gcc", "-std=c99", "-Wall", "-Werror", "-fsyntax-only", "-I", str(HEADER.parent), "-x", "c", "-"],
                       input=src, text=True, capture_output=True)
    assert r.returncode == 0, r.stderr


def test_every_declared_symbol_is_exported(library):
    names = _declared()
    assert len(names) >= 18
    missing = [n for n in names if not hasattr(library, n)]
    assert not missing, missing


def test_binding_lists_the_same_names():
    import paper_1609_06634_b200 as B
    assert sorted(B.EXPORTED_SYMBOLS) == _declared()
    methods = {n[len("bioem_"):] for n in _declared()} - {"create", "destroy", "last_error", "ctf_from_defocus"}
    missing = [m for m in methods if not hasattr(B.BioEM, m)]
    assert not missing, missing


def test_dynamic_symbol_table_has_no_cxx_mangled_api(library):
    import paper_1609_06634_b200 as B
    out = subprocess.run(["nm", "-D", "--defined-only", str(B.library_path())], capture_output=True, text=True).stdout
    exported = {ln.split()[-1] for ln in out.splitlines() if " T " in ln}
    assert set(_declared()) <= exported


def test_host_only_helper_and_error_paths(library):
    """bioem_ctf_from_defocus needs no device (R8/R9 constants): 1 um at 300 kV -> a = lambda_e dz / (2 pi)."""
    a, b = ctypes.c_float(), ctypes.c_float()
    assert library.bioem_ctf_from_defocus(1.0, 50.0, 300.0, ctypes.byref(a), ctypes.byref(b)) == 0
    golden = dict(ln.split()[:2] for ln in (ROOT / "tests" / "golden" / "ctf_constants.txt").read_text().splitlines()
                  if ln.strip() and not ln.startswith("#"))
    assert abs(a.value - float(golden["a_A2_1um_300kV"])) <= 2e-3
    assert abs(b.value - float(golden["b_A2_B50"])) <= 1e-5
    assert library.bioem_ctf_from_defocus(1.0, 50.0, -1.0, ctypes.byref(a), ctypes.byref(b)) != 0   # bad argument, no abort
    assert library.bioem_create(None, 0, None) != 0                                                # NULL out pointer


def test_noalloc_entry_point_checks_its_arguments_before_touching_the_device(library):
    """bioem_ensemble_log_posterior_noalloc: NULL pointers and sizes beyond the fixed work array are refused with a message and
    nothing is enqueued (the checks come before the first CUDA call, so they run here without a device)."""
    from paper_1609_06634_b200 import binding
    one = ctypes.c_void_p(8)                                       # never dereferenced: the calls below return before any launch
    f = library.bioem_ensemble_log_posterior_noalloc
    assert f(0, None, 4, 2, None, None, one, None) == -1
    assert f(0, None, 4, 2, one, None, None, None) == -1
    assert f(0, None, 0, 2, one, None, one, None) == -1
    assert f(0, None, binding.NOALLOC_MAX_IMG + 1, 2, one, None, one, None) == -5
    msg = library.bioem_noalloc_last_error().decode()
    assert str(binding.NOALLOC_MAX_IMG) in msg and "at most" in msg
    assert f(0, None, 4, binding.NOALLOC_MAX_MODEL + 1, one, None, one, None) == -5
    assert library.bioem_noalloc_prepare(-1) == -1 and library.bioem_noalloc_prepare(64) == -1
    header = HEADER.read_text()
    assert f"#define BIOEM_NOALLOC_MAX_IMG   {binding.NOALLOC_MAX_IMG}" in header
    assert f"#define BIOEM_NOALLOC_MAX_MODEL {binding.NOALLOC_MAX_MODEL}" in header


def test_no_device_means_loud_failure(library):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    from paper_1609_06634_b200 import BioEM, BioEMError
    with pytest.raises(BioEMError):
        BioEM()


def test_product_package_never_imports_the_oracle():
    for f in (ROOT / "paper_1609_06634_b200").rglob("*"):
        if f.suffix in (".py", ".cu", ".cuh", ".h"):
            assert "oracle" not in f.read_text().replace("test oracle", ""), f
