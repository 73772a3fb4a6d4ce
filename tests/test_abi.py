"""-m "not gpu": the C-ABI library builds for sm_100a, loads, and exports every symbol include/e2e.h declares.
No compute call is made here (there is no GPU); only argument validation that fails before any CUDA call."""
import ctypes as C
import re
import subprocess
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parent.parent


@pytest.fixture(scope="module")
def lib():
    from paper_2008_05858_b200 import build, binding
    build.build()
    return binding.load()


def _declared():
    text = (ROOT / "include" / "e2e.h").read_text()
    return sorted(set(re.findall(r"E2E_API\s+[\w\s\*]+?\b(e2e_\w+)\s*\(", text)))


def test_header_declares_the_north_star_entry_points():
    names = _declared()
    for n in ("e2e_format_create", "e2e_psf_create", "e2e_render_frame", "e2e_apply_detector"):
        assert n in names


def test_every_declared_symbol_is_exported(lib):
    from paper_2008_05858_b200 import binding
    names = _declared()
    assert sorted(binding.SYMBOLS) == names
    out = subprocess.run(["nm", "-D", "--defined-only", str(binding.LIB_PATH)], capture_output=True, text=True, check=True).stdout
    exported = set(re.findall(r" T (e2e_\w+)", out))
    assert exported == set(names)
    for n in names:
        assert getattr(lib, n) is not None


def test_library_holds_sm_100a_code():
    from paper_2008_05858_b200 import binding, build
    build.build()
    out = subprocess.run(["cuobjdump", "-lelf", str(binding.LIB_PATH)], capture_output=True, text=True).stdout
    assert "sm_100a" in out


def test_version_and_argument_validation_without_a_device(lib):
    from paper_2008_05858_b200 import binding
    assert "sm_100a" in binding.e2e_version()
    h = C.c_void_p()
    assert lib.e2e_format_create(C.byref(h), None) == -1
    assert "NULL" in binding.e2e_last_error()
    assert lib.e2e_psf_create(C.byref(h), None, 16, 16) == -1
    d = binding.PsfDesc()
    d.kind, d.sigma_x, d.sigma_y = 0, -1.0, 1.0
    assert lib.e2e_psf_create(C.byref(h), C.byref(d), 16, 16) == -1          # negative sigma
    d.kind = 7
    assert lib.e2e_psf_create(C.byref(h), C.byref(d), 16, 16) == -1          # unknown kind
    d.kind, d.sigma_x, d.fiber_dx_px = 0, 1.0, 200.0
    assert lib.e2e_psf_create(C.byref(h), C.byref(d), 16, 16) == -5          # footprint limit -> UNSUPPORTED
    assert lib.e2e_apply_detector(None, None, 4, 4, None, None) == -1
    assert lib.e2e_render_frame(None, None, None, None, 0, None, 0, None) == -1


def test_product_package_never_imports_the_oracle():
    for p in (ROOT / "paper_2008_05858_b200").rglob("*"):
        if p.suffix in (".py", ".cu", ".cuh", ".h") and p.is_file():
            t = p.read_text()
            assert "import oracle" not in t and "from oracle" not in t and "liboracle" not in t, p
