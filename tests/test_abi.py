"""-m "not gpu": the C-ABI shared library builds, loads and exports every function include/rism3d.h declares;
argument checks that need no device; the Python binding has the same names.  No compute calls here."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "rism3d.h")
HEADER_1D = os.path.join(ROOT, "include", "rism1d.h")


def declared_functions(header=HEADER, prefix="rism3d_"):
    """Names of the functions declared in a header of include/ (prototype = `name(` at the start of a declaration)."""
    src = open(header).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)          # drop comments
    names = re.findall(r"\b(" + prefix + r"[a-z0-9_]+)\s*\(", src)
    return sorted(set(names))


@pytest.fixture(scope="module")
def lib():
    from paper_2403_01039_b200 import build as _build
    _build.build(force=False)
    import paper_2403_01039_b200 as pkg
    return pkg


def test_header_declares_the_north_star_calls():
    names = declared_functions()
    for must in ("rism3d_init", "rism3d_set_solute", "rism3d_set_solvent_chi", "rism3d_iterate", "rism3d_free_energy"):
        assert must in names


def test_library_exports_every_declared_symbol(lib):
    handle = lib.load_library()
    for name in declared_functions():
        assert hasattr(handle, name), f"librism3d.so does not export {name}"
    # and the binding lists exactly the header's functions, each with a Python function of the same name
    assert sorted(lib.EXPORTED_SYMBOLS) == declared_functions()
    for name in declared_functions():
        assert callable(getattr(lib, name)), f"binding has no function {name}"


def test_library_exports_every_symbol_of_the_1d_header(lib):
    handle = lib.load_library()
    names = declared_functions(HEADER_1D, "rism1d_")
    assert "rism1d_solve" in names and "rism1d_get_chi" in names
    for name in names:
        assert hasattr(handle, name), f"librism3d.so does not export {name}"
        assert callable(getattr(lib, name)), f"binding has no function {name}"
    assert sorted(lib.EXPORTED_SYMBOLS_1D) == names
    p = lib.Rism1dParams()
    p.n_sites, p.n_points, p.dr, p.temperature, p.kappa, p.closure, p.pse_order = 3, 2048, 0.025, 298.0, 1.0, 1, 1
    p.mdiis_nvec, p.mdiis_b, p.mdiis_restart = 10, 0.5, 10.0
    assert lib.rism1d_workspace_bytes(p) > 0
    for field, bad in [("n_sites", 9), ("n_points", 1000), ("n_points", 32768), ("dr", 0.0), ("mdiis_nvec", 17)]:
        keep = getattr(p, field)
        setattr(p, field, bad)
        assert lib.rism1d_workspace_bytes(p) == 0
        setattr(p, field, keep)


def test_no_torch_types_in_the_abi():
    for header in (HEADER, HEADER_1D):
        src = open(header).read()
        code = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
        assert "torch" not in code.lower() and "at::" not in code and "#include <cuda" not in code
        assert 'extern "C"' in src


def test_workspace_bytes_and_argument_checks_without_a_device(lib):
    p = lib.Rism3dParams()
    p.nx = p.ny = p.nz = 64
    p.spacing = 0.5
    p.n_sites = 2
    p.closure = 1
    p.pse_order = 1
    p.temperature = 298.0
    p.mdiis_nvec = 5
    p.mdiis_b = 0.5
    p.mdiis_restart = 10.0
    p.kappa = 1.0
    p.r_min = 1e-3
    handle = lib.load_library()
    nbytes = handle.rism3d_workspace_bytes(C.byref(p))
    field = 64 ** 3 * 2 * 8
    # 2M history field-sets + tau + w + work + phi + phi~ and small tables
    assert (2 * 5 + 3 + 1) * field <= nbytes <= (2 * 5 + 3 + 1) * field + (8 << 20)
    p.nx = 48                                         # not a power of two
    assert handle.rism3d_workspace_bytes(C.byref(p)) == 0
    p.nx = 64
    p.n_sites = 3                                     # runs padded to 4 site types
    four = 64 ** 3 * 4 * 8
    assert (2 * 5 + 3) * four <= handle.rism3d_workspace_bytes(C.byref(p)) <= (2 * 5 + 3 + 1) * four + (8 << 20)
    p.n_sites = 9
    assert handle.rism3d_workspace_bytes(C.byref(p)) == 0
    p.n_sites = 2
    p.r_min = 0.0                                     # a zero-initialised clamp is refused
    assert handle.rism3d_workspace_bytes(C.byref(p)) == 0
    p.r_min = 1e-3
    p.mdiis_nvec = 17
    assert handle.rism3d_workspace_bytes(C.byref(p)) == 0
    # NULL context: every entry point answers with an error code instead of crashing
    assert handle.rism3d_iterate(None, 1, 0.0, None, None) == -1
    assert handle.rism3d_free_energy(None, None, None) == -1
    assert handle.rism3d_launch_count(None) == 0
    handle.rism3d_destroy(None)
    assert lib.rism3d_status_string(-8) == "iteration diverged"
    assert "barrier" in lib.rism3d_status_string(-9)
    # the IPC helpers take a device ordinal, not a context: one that does not exist is refused before any CUDA call on it
    ptr = C.c_void_p()
    assert handle.rism3d_peer_alloc(4096, 1024, C.byref(ptr)) == -1 and not ptr.value
    assert handle.rism3d_peer_free(-1, None) == -1
    assert handle.rism3d_peer_close(4096, None) == -1
    assert lib.rism3d_loop_kernel_name(0) != "" and lib.rism3d_loop_kernel_name(99) == ""


def test_init_fails_loudly_without_cuda(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("this check is for the CPU-only box")
    p = lib.Rism3dParams()
    p.nx = p.ny = p.nz = 16
    p.spacing, p.n_sites, p.closure, p.pse_order, p.temperature = 0.5, 2, 1, 1, 298.0
    p.mdiis_nvec, p.mdiis_b, p.mdiis_restart, p.kappa, p.r_min = 2, 0.5, 10.0, 1.0, 1e-3
    handle = lib.load_library()
    ctx = C.c_void_p()
    rc = handle.rism3d_init(C.byref(ctx), C.byref(p), C.c_void_p(256), 1 << 40, None)
    assert rc == -7 and not ctx.value                 # RISM3D_ERR_CUDA: there is no CPU fallback
    with pytest.raises(Exception):
        lib.Solver(16, 0.5, 2)


def test_product_path_does_not_import_the_oracle():
    """The package and its C sources never reference oracle/ (the oracle is test infrastructure)."""
    pkg = os.path.join(ROOT, "paper_2403_01039_b200")
    for dirpath, _, files in os.walk(pkg):
        if "build" in os.path.relpath(dirpath, pkg).split(os.sep)[:1] and dirpath != pkg:
            continue
        for fn in files:
            if fn.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, fn)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", text, flags=re.M), fn
    for fn in os.listdir(os.path.join(ROOT, "oracle")):
        if fn.endswith(".py"):
            text = open(os.path.join(ROOT, "oracle", fn)).read()
            assert "paper_2403_01039_b200" not in text.replace("`paper_2403_01039_b200/`", ""), fn
