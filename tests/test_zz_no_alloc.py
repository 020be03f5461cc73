"""rism3d_noalloc_free_energy (include/rism3d_noalloc.h) -- the free-energy sum for users who cannot hand the library a
workspace: a plug-in inside an MD / QM program whose memory pool already owns the whole GPU (a cudaMalloc there fails),
code that must not stall the device with cudaMalloc / cudaFree between other streams' work, an analysis step that was
only given tau, w and phi.  Its partial sums live in a fixed 148 KiB `static __device__` array of the library image
instead of a caller-allocated workspace; limits: 8 site types, 512^3 points; one array per GPU, shared by every call.

This file is named so that pytest collects it LAST (`pytest --collect-only -q tests`): `-x` stops at the first failure,
and a failure here must not hide the parity tests.  The GPU test passes alone in a fresh process and after the others:
it depends on nothing the other tests leave behind, and the entry point itself must not care what the array holds.
"""
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "rism3d_noalloc.h")

FE_RTOL = 1e-7          # the suite's bar on a free energy (tests/test_gpu_parity.py, north_star "relative 1e-7")


def test_header_symbol_is_exported_and_bound():
    """-m "not gpu": the library exports what include/rism3d_noalloc.h declares, the binding has the same name and the
    same limits, and the source of the entry point contains no allocating call."""
    from paper_2403_01039_b200 import build as _build
    _build.build(force=False)
    import paper_2403_01039_b200 as lib
    src = re.sub(r"/\*.*?\*/", "", open(HEADER).read(), flags=re.S)
    names = sorted(set(re.findall(r"\b(rism3d_[a-z0-9_]+)\s*\(", src)))
    assert names == sorted(lib.EXPORTED_SYMBOLS_NOALLOC) == ["rism3d_noalloc_free_energy"]      # ONE entry point
    handle = lib.load_library()
    for name in names:
        assert hasattr(handle, name) and callable(getattr(lib, name))
    defs = dict(re.findall(r"#define\s+(RISM3D_NOALLOC_[A-Z_]+)\s+(\d+)", src))
    assert int(defs["RISM3D_NOALLOC_MAX_SITES"]) == lib.NOALLOC_MAX_SITES == 8
    assert int(defs["RISM3D_NOALLOC_MAX_POINTS"]) == lib.NOALLOC_MAX_POINTS == 512 ** 3
    assert int(defs["RISM3D_NOALLOC_SCRATCH_BYTES"]) == lib.NOALLOC_SCRATCH_BYTES == 2 * 592 * 8 * 2 * 8
    code = open(os.path.join(ROOT, "paper_2403_01039_b200", "csrc", "noalloc.cu")).read()
    code = re.sub(r"//[^\n]*", "", code)                      # comments may name what the code must not call
    assert not re.search(r"cudaMalloc|cudaFree|cudaHostAlloc|cudaMemPool|\bmalloc\s*\(|\bnew\b|std::vector", code)
    assert "cudaGetSymbolAddress" in code


def test_argument_checks_need_no_device():
    """Sizes beyond the fixed array are refused with a message, before anything touches a GPU."""
    import paper_2403_01039_b200 as lib
    one = np.ones(1)
    ok = dict(device=0, cuda_stream=0, n_points=64, spacing=0.5, n_sites=1, closure=1, pse_order=1, temperature=298.0,
              q=one, rho=one, d_tau=256, d_w=256, d_phi=256, d_out=256)       # dummy non-NULL addresses: never dereferenced
    for change, status, word in [
        (dict(n_sites=9, q=np.ones(9), rho=np.ones(9)), -2, "n_sites = 9"),
        (dict(n_points=512 ** 3 + 1), -2, "n_points"),
        (dict(n_points=0), -2, "n_points"),
        (dict(spacing=0.0), -2, "positive"),
        (dict(closure=7), -1, "closure"),
        (dict(d_out=0), -1, "NULL"),
    ]:
        with pytest.raises(lib.Rism3dError) as ei:
            lib.rism3d_noalloc_free_energy(**{**ok, **change})
        assert ei.value.status == status and word in str(ei.value), str(ei.value)


def _solved(lib, n, solvent, closure, pse_order, n_iter):
    """A solver of the existing (workspace) path after n_iter iterations, and what it reports."""
    from workloads import load_chi, make_solute, solvent_by_name
    sv = solvent_by_name(solvent)
    sol = make_solute("C1")
    k0, dk, chi = load_chi(sv.name)
    s = lib.Solver(n, 0.5, sv.n_v, closure=closure, pse_order=pse_order, mdiis_nvec=5)
    s.set_solvent_chi(sv.q, sv.sigma, sv.eps, sv.rho, k0, dk, chi)
    s.set_solute(sol.xyz, sol.q, sol.sigma, sol.eps)
    s.iterate(n_iter, 0.0)
    mu, mu_site = s.free_energy()                     # rism3d_free_energy: partial sums in the caller's workspace
    _, c_int = s.pmv(1.0)                             # per-site dV sum c_sr of the same kernel
    return s, sv, mu, mu_site, c_int


def _fields_on_device(torch, s):
    tau = torch.stack([s.get_field_device("TAU", g) for g in range(s.n_sites)]).reshape(s.n_sites, -1).contiguous()
    w = torch.stack([s.get_field_device("W", g) for g in range(s.n_sites)]).reshape(s.n_sites, -1).contiguous()
    phi = s.get_field_device("PHI", 0).reshape(-1).contiguous()
    s.stream.synchronize()
    torch.cuda.synchronize()
    return tau, w, phi


@pytest.mark.gpu
def test_noalloc_free_energy_matches_the_workspace_path_on_consecutive_calls():
    """Two solved states with different site counts, closures and grids; the no-allocation entry point is called for
    the 4-site one, then at once for the 2-site one (which leaves the first call's values in the upper slots of the
    shared array), then for the first again -- all on one stream, no synchronisation in between -- and every result is
    held to what rism3d_free_energy / rism3d_pmv of the existing path returned for the same fields."""
    import torch
    import paper_2403_01039_b200 as lib
    dev = torch.device("cuda", 0)
    a = _solved(lib, 32, "water_nacl_0.1M", "PSE", 2, 12)
    b = _solved(lib, 64, "water", "KH", 1, 20)
    cases = []
    for s, sv, mu, mu_site, c_int in (a, b):
        tau, w, phi = _fields_on_device(torch, s)
        out = torch.full((2, s.n_sites), float("nan"), dtype=torch.float64, device=dev)
        cases.append((s, sv, mu, mu_site, c_int, tau, w, phi, out))
    third = torch.full((2, a[0].n_sites), float("nan"), dtype=torch.float64, device=dev)
    torch.cuda.synchronize()
    allocated = torch.cuda.memory_allocated(dev)

    stream = torch.cuda.Stream(dev)
    calls = [(cases[0], cases[0][8]), (cases[1], cases[1][8]), (cases[0], third)]
    for (s, sv, _, _, _, tau, w, phi, _), out in calls:           # back to back, ordered by the stream only
        lib.rism3d_noalloc_free_energy(0, stream.cuda_stream, tau.shape[1], s.spacing, s.n_sites,
                                       s.params.closure, s.params.pse_order, s.params.temperature, sv.q, sv.rho,
                                       tau.data_ptr(), w.data_ptr(), phi.data_ptr(), out.data_ptr())
    stream.synchronize()
    assert torch.cuda.memory_allocated(dev) == allocated          # torch's view; the C side has no allocating call at all

    for (s, sv, mu, mu_site, c_int, *_), out in calls:
        got = out.cpu().numpy()
        assert np.all(np.isfinite(got))
        assert abs(got[0].sum() - mu) <= FE_RTOL * abs(mu), (got[0].sum(), mu)
        np.testing.assert_allclose(got[0], mu_site, rtol=FE_RTOL, atol=FE_RTOL * abs(mu))
        np.testing.assert_allclose(got[1], c_int, rtol=FE_RTOL, atol=FE_RTOL * np.max(np.abs(c_int)))
    assert torch.equal(cases[0][8], third)                        # same inputs, same fixed summation order: same bits
    for s, *_ in cases:
        s.close()
