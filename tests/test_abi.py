"""The C-ABI library loads on a CPU-only box and exports every symbol include/cola.h declares; argument
validation that needs no GPU returns the documented status codes.  No compute calls here."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2302_00850_b200 import build

    path = build.build()
    return ctypes.CDLL(path)


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "cola.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(cola_[a-z0-9_]+)\s*\(", text)))


def test_header_declares_the_north_star_entry_points():
    syms = declared_symbols()
    for name in ("cola_gauge_upload", "cola_dslash_apply", "cola_fermion_matrix_apply", "cola_schur_apply", "cola_cg_solve"):
        assert name in syms


def test_library_exports_every_declared_symbol(lib):
    syms = declared_symbols()
    assert len(syms) >= 20
    for name in syms:
        assert hasattr(lib, name), f"libcola.so does not export {name}"


def test_binding_lists_the_same_names(lib):
    from paper_2302_00850_b200 import binding

    assert sorted(binding.EXPORTS) == declared_symbols()
    for name in binding.EXPORTS:
        method = name[len("cola_"):]
        if method in ("create", "destroy", "last_error"):
            continue
        if method in ("selftest_host", "spinor_norm2_static"):   # context-free: module-level functions
            assert hasattr(binding, method)
            continue
        assert hasattr(binding.Cola, method), f"binding lacks Cola.{method}"


def test_create_rejects_bad_lattices_without_touching_the_gpu(lib):
    from paper_2302_00850_b200 import binding

    lib.cola_last_error.restype = ctypes.c_char_p
    lib.cola_last_error.argtypes = [ctypes.c_void_p]
    for dims, bc in (((3, 4, 4, 4), (1, 1, 1, -1)), ((4, 4, 4, 0), (1, 1, 1, -1)), ((4, 4, 4, 4), (1, 1, 1, 0))):
        p = binding.ColaParams()
        p.dims[:] = dims
        p.bc[:] = bc
        p.kappa, p.csw = 0.12, 1.0
        h = ctypes.c_void_p()
        st = lib.cola_create(ctypes.byref(h), ctypes.byref(p))
        assert st == binding.COLA_EINVAL
        assert not h.value
        assert b"cola_create" in lib.cola_last_error(None)
    # largest lattice: site indices are 32-bit, so a half volume above 2e9 is refused (1024^3 x 8 = 4.3e9 per parity)
    p = binding.ColaParams()
    p.dims[:] = (1024, 1024, 1024, 8)
    p.bc[:] = (1, 1, 1, -1)
    h = ctypes.c_void_p()
    assert lib.cola_create(ctypes.byref(h), ctypes.byref(p)) == binding.COLA_EINVAL and not h.value
    assert b"32-bit" in lib.cola_last_error(None)
    assert lib.cola_create(None, None) == binding.COLA_EINVAL
    assert lib.cola_destroy(None) == binding.COLA_OK


def test_oracle_and_cuda_path_share_no_code():
    """The oracle must not include or import the product, and vice versa."""
    for d, banned in (("oracle", ("paper_2302_00850_b200", "csrc", "cola.h")), ("paper_2302_00850_b200", ("oracle",))):
        for base, _, files in os.walk(os.path.join(ROOT, d)):
            for f in files:
                if not f.endswith((".py", ".c", ".h", ".cu", ".cuh")):
                    continue
                text = open(os.path.join(base, f)).read()
                for line in text.splitlines():
                    s = line.strip()
                    if s.startswith(("import ", "from ", "#include")):
                        for b in banned:
                            assert b not in s, f"{d}/{f}: '{s}'"


def test_host_index_machinery_selftest(lib):
    """Magic-number division vs hardware division for every divisor <= 4200, tile shapes, sweep permutations (no GPU)."""
    from paper_2302_00850_b200 import binding

    assert binding.selftest_host() == "ok"
