"""ctypes binding of librism3d.so -- same names as include/rism3d.h, argument marshalling only.

`Solver` is a thin convenience object that owns the device workspace (a torch uint8 tensor) and the
opaque context; every method is one C call.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB = None

CLOSURES = {"KH": 1, "PSE": 2, "HNC": 3}
ACCELERATORS = {"MDIIS": 0, "ANDERSON": 1}
FIELDS = {"G": 0, "H": 1, "C_SR": 2, "T": 3, "TAU": 4, "W": 5, "PHI": 6}

EXPORTED_SYMBOLS = [
    "rism3d_workspace_bytes", "rism3d_init", "rism3d_set_solvent_chi", "rism3d_set_solute",
    "rism3d_iterate", "rism3d_free_energy", "rism3d_pmv", "rism3d_pressure_correction", "rism3d_gradient", "rism3d_get_field", "rism3d_set_tau",
    "rism3d_get_rms_history", "rism3d_launch_count", "rism3d_phi_ms", "rism3d_measure_dfma_peak", "rism3d_set_profiling", "rism3d_get_timings",
    "rism3d_loop_kernel_name", "rism3d_debug_fft_forward",
    "rism3d_debug_fft_inverse", "rism3d_last_error", "rism3d_status_string", "rism3d_destroy",
    "rism3d_slab_plan", "rism3d_slab_local", "rism3d_slab_set_peers", "rism3d_slab_begin", "rism3d_slab_phase",
    "rism3d_slab_status", "rism3d_slab_end", "rism3d_slab_set_peer_timeout", "rism3d_debug_peer_barrier_selftest",
    "rism3d_slab_combine",
    "rism3d_peer_alloc", "rism3d_peer_free", "rism3d_peer_export", "rism3d_peer_open", "rism3d_peer_close",
]
EXPORTED_SYMBOLS_1D = [
    "rism1d_workspace_bytes", "rism1d_init", "rism1d_set_solvent", "rism1d_solve", "rism1d_get_pair", "rism1d_get_chi",
    "rism1d_get_chi_types", "rism1d_thermo", "rism1d_launch_count", "rism1d_last_error", "rism1d_destroy",
]
EXPORTED_SYMBOLS_NOALLOC = ["rism3d_noalloc_free_energy"]          # include/rism3d_noalloc.h
NOALLOC_MAX_SITES, NOALLOC_MAX_POINTS, NOALLOC_SCRATCH_BYTES = 8, 134217728, 151552


class Rism3dError(RuntimeError):
    def __init__(self, status: int, message: str):
        super().__init__(f"rism3d status {status}: {message}")
        self.status = status


class Rism3dParams(C.Structure):
    _fields_ = [
        ("nx", C.c_int), ("ny", C.c_int), ("nz", C.c_int),
        ("spacing", C.c_double),
        ("origin", C.c_double * 3),
        ("n_sites", C.c_int),
        ("closure", C.c_int),
        ("pse_order", C.c_int),
        ("temperature", C.c_double),
        ("mdiis_nvec", C.c_int),
        ("mdiis_b", C.c_double),
        ("mdiis_restart", C.c_double),
        ("kappa", C.c_double),
        ("r_min", C.c_double),
        ("device", C.c_int),
        ("accelerator", C.c_int),
        ("anderson_s", C.c_double * 2),
        ("mdiis_dynamic_b", C.c_int),
        ("mdiis_b_min", C.c_double), ("mdiis_b_max", C.c_double),
        ("n_ranks", C.c_int), ("rank", C.c_int),
    ]


class Rism1dParams(C.Structure):
    _fields_ = [("n_sites", C.c_int), ("n_points", C.c_int), ("dr", C.c_double), ("temperature", C.c_double),
                ("kappa", C.c_double), ("closure", C.c_int), ("pse_order", C.c_int), ("mdiis_nvec", C.c_int),
                ("mdiis_b", C.c_double), ("mdiis_restart", C.c_double), ("device", C.c_int)]


class Rism3dSlabInfo(C.Structure):
    _fields_ = [("nxl", C.c_int), ("ix0", C.c_int), ("nyl", C.c_int), ("jy0", C.c_int), ("n_sites_padded", C.c_int),
                ("row_elems", C.c_size_t), ("block_elems", C.c_size_t)]


def library_path() -> str:
    return os.path.join(_HERE, "librism3d.so")


def load_library():
    """Load librism3d.so; raises (never falls back) when it has not been built."""
    global _LIB
    if _LIB is not None:
        return _LIB
    path = library_path()
    if not os.path.exists(path):
        raise RuntimeError(f"{path} not found: build it with `python -m paper_2403_01039_b200.build` "
                           "(there is no CPU fallback)")
    lib = C.CDLL(path)
    dp, ip = C.POINTER(C.c_double), C.POINTER(C.c_int)
    lib.rism3d_workspace_bytes.restype = C.c_size_t
    lib.rism3d_workspace_bytes.argtypes = [C.POINTER(Rism3dParams)]
    lib.rism3d_init.restype = C.c_int
    lib.rism3d_init.argtypes = [C.POINTER(C.c_void_p), C.POINTER(Rism3dParams), C.c_void_p, C.c_size_t, C.c_void_p]
    lib.rism3d_set_solvent_chi.restype = C.c_int
    lib.rism3d_set_solvent_chi.argtypes = [C.c_void_p, dp, dp, dp, dp, C.c_int, C.c_double, C.c_double, dp]
    lib.rism3d_set_solute.restype = C.c_int
    lib.rism3d_set_solute.argtypes = [C.c_void_p, C.c_int, dp, dp, dp, dp, C.c_double, C.POINTER(C.c_float)]
    lib.rism3d_iterate.restype = C.c_int
    lib.rism3d_iterate.argtypes = [C.c_void_p, C.c_int, C.c_double, ip, dp]
    lib.rism3d_free_energy.restype = C.c_int
    lib.rism3d_free_energy.argtypes = [C.c_void_p, dp, dp]
    lib.rism3d_pmv.restype = C.c_int
    lib.rism3d_pmv.argtypes = [C.c_void_p, C.c_double, dp, dp]
    lib.rism3d_pressure_correction.restype = C.c_int
    lib.rism3d_pressure_correction.argtypes = [C.c_void_p, C.c_double, C.c_double, dp, dp]
    lib.rism3d_gradient.restype = C.c_int
    lib.rism3d_gradient.argtypes = [C.c_void_p, dp]
    lib.rism3d_measure_dfma_peak.restype = C.c_int
    lib.rism3d_measure_dfma_peak.argtypes = [C.c_void_p, dp]
    lib.rism3d_phi_ms.restype = C.c_int
    lib.rism3d_phi_ms.argtypes = [C.c_void_p, C.POINTER(C.c_float)]
    lib.rism3d_get_field.restype = C.c_int
    lib.rism3d_get_field.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_void_p, C.c_int]
    lib.rism3d_set_tau.restype = C.c_int
    lib.rism3d_set_tau.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_int]
    lib.rism3d_get_rms_history.restype = C.c_int
    lib.rism3d_get_rms_history.argtypes = [C.c_void_p, dp, C.c_int, ip]
    lib.rism3d_launch_count.restype = C.c_longlong
    lib.rism3d_launch_count.argtypes = [C.c_void_p]
    lib.rism3d_set_profiling.restype = C.c_int
    lib.rism3d_set_profiling.argtypes = [C.c_void_p, C.c_int]
    lib.rism3d_get_timings.restype = C.c_int
    lib.rism3d_get_timings.argtypes = [C.c_void_p, dp, C.c_int, C.POINTER(C.c_longlong)]
    lib.rism3d_loop_kernel_name.restype = C.c_char_p
    lib.rism3d_loop_kernel_name.argtypes = [C.c_int]
    lib.rism3d_debug_fft_forward.restype = C.c_int
    lib.rism3d_debug_fft_forward.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
    lib.rism3d_debug_fft_inverse.restype = C.c_int
    lib.rism3d_debug_fft_inverse.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
    lib.rism3d_last_error.restype = C.c_char_p
    lib.rism3d_last_error.argtypes = [C.c_void_p]
    lib.rism3d_status_string.restype = C.c_char_p
    lib.rism3d_status_string.argtypes = [C.c_int]
    lib.rism3d_destroy.restype = None
    lib.rism3d_destroy.argtypes = [C.c_void_p]
    vpp, szp = C.POINTER(C.c_void_p), C.POINTER(C.c_size_t)
    lib.rism3d_slab_plan.restype = C.c_int
    lib.rism3d_slab_plan.argtypes = [C.POINTER(Rism3dParams), C.POINTER(Rism3dSlabInfo)]
    lib.rism3d_slab_local.restype = C.c_int
    lib.rism3d_slab_local.argtypes = [C.c_void_p, vpp, vpp, vpp, vpp, szp, szp]
    lib.rism3d_slab_set_peers.restype = C.c_int
    lib.rism3d_slab_set_peers.argtypes = [C.c_void_p, vpp, vpp, vpp]
    lib.rism3d_slab_set_peer_timeout.restype = C.c_int
    lib.rism3d_slab_set_peer_timeout.argtypes = [C.c_void_p, C.c_double]
    lib.rism3d_debug_peer_barrier_selftest.restype = C.c_int
    lib.rism3d_debug_peer_barrier_selftest.argtypes = [C.c_int, C.c_void_p, C.c_size_t, C.c_void_p, C.c_int, C.c_int, C.c_int,
                                                       C.c_double, ip, ip]
    lib.rism3d_slab_combine.restype = C.c_int
    lib.rism3d_slab_combine.argtypes = [dp, C.c_int, C.c_int, dp]
    lib.rism3d_slab_begin.restype = C.c_int
    lib.rism3d_slab_begin.argtypes = [C.c_void_p, C.c_double]
    lib.rism3d_slab_phase.restype = C.c_int
    lib.rism3d_slab_phase.argtypes = [C.c_void_p, C.c_int]
    lib.rism3d_slab_status.restype = C.c_int
    lib.rism3d_slab_status.argtypes = [C.c_void_p, ip, ip, dp]
    lib.rism3d_slab_end.restype = C.c_int
    lib.rism3d_slab_end.argtypes = [C.c_void_p, ip, dp]
    lib.rism3d_peer_alloc.restype = C.c_int
    lib.rism3d_peer_alloc.argtypes = [C.c_int, C.c_size_t, vpp]
    lib.rism3d_peer_free.restype = C.c_int
    lib.rism3d_peer_free.argtypes = [C.c_int, C.c_void_p]
    lib.rism3d_peer_export.restype = C.c_int
    lib.rism3d_peer_export.argtypes = [C.c_int, C.c_void_p, C.POINTER(C.c_ubyte)]
    lib.rism3d_peer_open.restype = C.c_int
    lib.rism3d_peer_open.argtypes = [C.c_int, C.POINTER(C.c_ubyte), vpp]
    lib.rism3d_peer_close.restype = C.c_int
    lib.rism3d_peer_close.argtypes = [C.c_int, C.c_void_p]
    # ---- include/rism1d.h ----
    lib.rism1d_workspace_bytes.restype = C.c_size_t
    lib.rism1d_workspace_bytes.argtypes = [C.POINTER(Rism1dParams)]
    lib.rism1d_init.restype = C.c_int
    lib.rism1d_init.argtypes = [C.POINTER(C.c_void_p), C.POINTER(Rism1dParams), C.c_void_p, C.c_size_t, C.c_void_p]
    lib.rism1d_set_solvent.restype = C.c_int
    lib.rism1d_set_solvent.argtypes = [C.c_void_p, dp, dp, dp, dp, ip, dp]
    lib.rism1d_solve.restype = C.c_int
    lib.rism1d_solve.argtypes = [C.c_void_p, C.c_double, C.c_int, C.c_double, ip, dp]
    lib.rism1d_get_pair.restype = C.c_int
    lib.rism1d_get_pair.argtypes = [C.c_void_p, C.c_int, dp]
    lib.rism1d_get_chi.restype = C.c_int
    lib.rism1d_get_chi.argtypes = [C.c_void_p, dp]
    lib.rism1d_get_chi_types.restype = C.c_int
    lib.rism1d_get_chi_types.argtypes = [C.c_void_p, C.c_int, ip, dp]
    lib.rism1d_thermo.restype = C.c_int
    lib.rism1d_thermo.argtypes = [C.c_void_p, dp, dp, dp]
    lib.rism1d_launch_count.restype = C.c_longlong
    lib.rism1d_launch_count.argtypes = [C.c_void_p]
    lib.rism1d_last_error.restype = C.c_char_p
    lib.rism1d_last_error.argtypes = [C.c_void_p]
    lib.rism1d_destroy.restype = None
    lib.rism1d_destroy.argtypes = [C.c_void_p]
    # rism3d_noalloc.h
    lib.rism3d_noalloc_free_energy.restype = C.c_int
    lib.rism3d_noalloc_free_energy.argtypes = [C.c_int, C.c_void_p, C.c_size_t, C.c_double, C.c_int, C.c_int, C.c_int,
                                               C.c_double, dp, dp, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p,
                                               C.c_char_p, C.c_size_t]
    _LIB = lib
    return lib


def _dptr(a: np.ndarray):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _f64(a) -> np.ndarray:
    return np.ascontiguousarray(np.asarray(a, dtype=np.float64))


def _check(ctx, status: int):
    if status != 0:
        lib = load_library()
        msg = lib.rism3d_last_error(ctx).decode() if ctx else ""
        raise Rism3dError(status, msg or lib.rism3d_status_string(status).decode())


# ---- the C calls, one Python function each -------------------------------------------------------
def rism3d_status_string(status: int) -> str:
    return load_library().rism3d_status_string(int(status)).decode()


def rism3d_last_error(ctx) -> str:
    return load_library().rism3d_last_error(ctx).decode()


def rism3d_workspace_bytes(params: Rism3dParams) -> int:
    return int(load_library().rism3d_workspace_bytes(C.byref(params)))


def rism3d_init(params: Rism3dParams, d_workspace: int, nbytes: int, cuda_stream: int):
    ctx = C.c_void_p()
    st = load_library().rism3d_init(C.byref(ctx), C.byref(params), C.c_void_p(d_workspace), nbytes,
                                    C.c_void_p(cuda_stream))
    if st != 0:
        raise Rism3dError(st, rism3d_status_string(st))
    return ctx


def rism3d_set_solvent_chi(ctx, q, sigma, eps, rho, k0: float, dk: float, chi):
    q, sigma, eps, rho, chi = _f64(q), _f64(sigma), _f64(eps), _f64(rho), _f64(chi)
    _check(ctx, load_library().rism3d_set_solvent_chi(ctx, _dptr(q), _dptr(sigma), _dptr(eps), _dptr(rho),
                                                      int(chi.shape[0]), float(dk), float(k0), _dptr(chi)))


def rism3d_set_solute(ctx, xyz, q, sigma, eps, rcut: float = 0.0) -> float:
    xyz, q, sigma, eps = _f64(xyz), _f64(q), _f64(sigma), _f64(eps)
    ms = C.c_float(0.0)
    _check(ctx, load_library().rism3d_set_solute(ctx, int(len(q)), _dptr(xyz), _dptr(q), _dptr(sigma), _dptr(eps),
                                                 float(rcut), C.byref(ms)))
    return float(ms.value)


def rism3d_iterate(ctx, max_iter: int, tol: float = 0.0):
    n, rms = C.c_int(0), C.c_double(0.0)
    _check(ctx, load_library().rism3d_iterate(ctx, int(max_iter), float(tol), C.byref(n), C.byref(rms)))
    return int(n.value), float(rms.value)


def rism3d_free_energy(ctx, n_sites: int):
    tot = C.c_double(0.0)
    site = np.zeros(n_sites)
    _check(ctx, load_library().rism3d_free_energy(ctx, C.byref(tot), _dptr(site)))
    return float(tot.value), site


def rism3d_noalloc_free_energy(device: int, cuda_stream: int, n_points: int, spacing: float, n_sites: int, closure: int,
                               pse_order: int, temperature: float, q, rho, d_tau: int, d_w: int, d_phi: int, d_out: int):
    """The free-energy sum for callers that cannot give the library a workspace (their host program's pool owns the
    whole GPU, or they must not stall the device with cudaMalloc / cudaFree): the partial sums live in a fixed 148 KiB
    array inside the library image, so this call allocates nothing.  d_tau, d_w: device addresses of
    [n_sites][n_points] doubles, d_phi: [n_points], d_out: [2][n_sites] (dmu per site in kcal/mol, then dV sum c_sr in
    A^3).  Enqueued on `cuda_stream` (a cudaStream_t as an integer, 0 = default stream) and NOT waited for.  At most 8
    site types and 512^3 points; one array per GPU shared by all calls -- calls that overlap on one GPU race.  Make
    the first call on each device during start-up, outside stream capture (include/rism3d_noalloc.h)."""
    q, rho = _f64(q), _f64(rho)
    if q.shape != (int(n_sites),) or rho.shape != (int(n_sites),):
        raise ValueError(f"q and rho must have shape ({int(n_sites)},), got {q.shape} and {rho.shape}")
    err = C.create_string_buffer(512)
    st = load_library().rism3d_noalloc_free_energy(int(device), C.c_void_p(cuda_stream), int(n_points), float(spacing),
                                                   int(n_sites), int(closure), int(pse_order), float(temperature),
                                                   _dptr(q), _dptr(rho), C.c_void_p(d_tau), C.c_void_p(d_w),
                                                   C.c_void_p(d_phi), C.c_void_p(d_out), err, len(err))
    if st != 0:
        raise Rism3dError(st, err.value.decode() or rism3d_status_string(st))


def rism3d_pmv(ctx, chi_t: float, n_sites: int):
    """-> (pmv in A^3, per-site integrals of c_sr in A^3)"""
    v = C.c_double(0.0)
    site = np.zeros(n_sites)
    _check(ctx, load_library().rism3d_pmv(ctx, float(chi_t), C.byref(v), _dptr(site)))
    return float(v.value), site


def rism3d_pressure_correction(ctx, chi_t: float, pressure: float):
    """-> (dmu_PC in kcal/mol, pmv in A^3)"""
    pc, v = C.c_double(0.0), C.c_double(0.0)
    _check(ctx, load_library().rism3d_pressure_correction(ctx, float(chi_t), float(pressure), C.byref(pc), C.byref(v)))
    return float(pc.value), float(v.value)


def rism3d_gradient(ctx, n_atoms: int) -> np.ndarray:
    """-> d(dmu)/dR [n_atoms][3], kcal/(mol A)"""
    out = np.zeros((n_atoms, 3))
    _check(ctx, load_library().rism3d_gradient(ctx, _dptr(out)))
    return out


def rism3d_measure_dfma_peak(ctx) -> float:
    tf = C.c_double(0.0)
    _check(ctx, load_library().rism3d_measure_dfma_peak(ctx, C.byref(tf)))
    return float(tf.value)


def rism3d_phi_ms(ctx) -> float:
    ms = C.c_float(0.0)
    _check(ctx, load_library().rism3d_phi_ms(ctx, C.byref(ms)))
    return float(ms.value)


def rism3d_get_field(ctx, which: int, site: int, dst_ptr: int, dst_is_device: bool):
    _check(ctx, load_library().rism3d_get_field(ctx, int(which), int(site), C.c_void_p(dst_ptr), int(dst_is_device)))


def rism3d_set_tau(ctx, site: int, src_ptr: int, src_is_device: bool):
    _check(ctx, load_library().rism3d_set_tau(ctx, int(site), C.c_void_p(src_ptr), int(src_is_device)))


def rism3d_get_rms_history(ctx, cap: int = 65536) -> np.ndarray:
    buf = np.zeros(cap)
    n = C.c_int(0)
    _check(ctx, load_library().rism3d_get_rms_history(ctx, _dptr(buf), cap, C.byref(n)))
    return buf[: n.value].copy()


def rism3d_launch_count(ctx) -> int:
    return int(load_library().rism3d_launch_count(ctx))


N_LOOP_KERNELS = 5


def rism3d_set_profiling(ctx, enable: bool):
    _check(ctx, load_library().rism3d_set_profiling(ctx, int(bool(enable))))


def rism3d_get_timings(ctx):
    """-> (ms_total[N_LOOP_KERNELS], n_iterations)"""
    ms = np.zeros(N_LOOP_KERNELS)
    n = C.c_longlong(0)
    _check(ctx, load_library().rism3d_get_timings(ctx, _dptr(ms), N_LOOP_KERNELS, C.byref(n)))
    return ms, int(n.value)


def rism3d_loop_kernel_name(k: int) -> str:
    return load_library().rism3d_loop_kernel_name(int(k)).decode()


def rism3d_debug_fft_forward(ctx, d_in: int, d_out: int):
    _check(ctx, load_library().rism3d_debug_fft_forward(ctx, C.c_void_p(d_in), C.c_void_p(d_out)))


def rism3d_debug_fft_inverse(ctx, d_in: int, d_out: int):
    _check(ctx, load_library().rism3d_debug_fft_inverse(ctx, C.c_void_p(d_in), C.c_void_p(d_out)))


def rism3d_slab_plan(params: Rism3dParams) -> Rism3dSlabInfo:
    """host-only (no GPU): the slab of rank params.rank"""
    info = Rism3dSlabInfo()
    st = load_library().rism3d_slab_plan(C.byref(params), C.byref(info))
    if st != 0:
        raise Rism3dError(st, rism3d_status_string(st))
    return info


def rism3d_slab_local(ctx):
    """-> dict(K, stage, gram, flags: device addresses; block_bytes, gram_row_bytes)"""
    k, stg, gr, fl = C.c_void_p(), C.c_void_p(), C.c_void_p(), C.c_void_p()
    bb, gb = C.c_size_t(), C.c_size_t()
    _check(ctx, load_library().rism3d_slab_local(ctx, C.byref(k), C.byref(stg), C.byref(gr), C.byref(fl), C.byref(bb), C.byref(gb)))
    return dict(K=k.value, stage=stg.value, gram=gr.value, flags=fl.value, block_bytes=bb.value, gram_row_bytes=gb.value)


def rism3d_slab_set_peers(ctx, d_K, d_gram, d_flags):
    n = len(d_K)
    arr = lambda v: (C.c_void_p * n)(*[int(x) for x in v])
    _check(ctx, load_library().rism3d_slab_set_peers(ctx, arr(d_K), arr(d_gram), arr(d_flags)))


def rism3d_slab_combine(per_rank) -> np.ndarray:
    """[n_ranks][n_values] shares of the ranks -> their sums in rank order (the addition happens in the library)"""
    rows = _f64(per_rank)
    if rows.ndim != 2:
        raise ValueError(f"per_rank must be [n_ranks][n_values], got shape {rows.shape}")
    out = np.zeros(rows.shape[1])
    st = load_library().rism3d_slab_combine(_dptr(rows), int(rows.shape[0]), int(rows.shape[1]), _dptr(out))
    if st != 0:
        raise Rism3dError(st, rism3d_status_string(st))
    return out


def rism3d_slab_set_peer_timeout(ctx, seconds: float):
    _check(ctx, load_library().rism3d_slab_set_peer_timeout(ctx, float(seconds)))


def rism3d_debug_peer_barrier_selftest(device: int, d_scratch: int, nbytes: int, cuda_stream: int, n_ranks: int, epochs: int,
                                       absent_rank: int = -1, timeout_s: float = 5.0):
    """-> (ordering errors, ranks that timed out) of the peer-mode barrier run as ONE cooperative launch on one GPU"""
    ne, nt = C.c_int(-1), C.c_int(-1)
    st = load_library().rism3d_debug_peer_barrier_selftest(int(device), C.c_void_p(d_scratch), int(nbytes),
                                                           C.c_void_p(cuda_stream), int(n_ranks), int(epochs),
                                                           int(absent_rank), float(timeout_s), C.byref(ne), C.byref(nt))
    if st != 0:
        raise Rism3dError(st, rism3d_status_string(st))
    return int(ne.value), int(nt.value)


def rism3d_peer_alloc(device: int, nbytes: int) -> int:
    ptr = C.c_void_p()
    st = load_library().rism3d_peer_alloc(int(device), int(nbytes), C.byref(ptr))
    if st != 0:
        raise Rism3dError(st, f"cudaMalloc of {nbytes} bytes failed")
    return ptr.value


def rism3d_peer_free(device: int, ptr: int):
    load_library().rism3d_peer_free(int(device), C.c_void_p(ptr))


def rism3d_peer_export(device: int, ptr: int) -> bytes:
    h = (C.c_ubyte * 64)()
    st = load_library().rism3d_peer_export(int(device), C.c_void_p(ptr), h)
    if st != 0:
        raise Rism3dError(st, "cudaIpcGetMemHandle failed")
    return bytes(h)


def rism3d_peer_open(device: int, handle: bytes) -> int:
    h = (C.c_ubyte * 64).from_buffer_copy(handle)
    ptr = C.c_void_p()
    st = load_library().rism3d_peer_open(int(device), h, C.byref(ptr))
    if st != 0:
        raise Rism3dError(st, "cudaIpcOpenMemHandle failed")
    return ptr.value


def rism3d_peer_close(device: int, ptr: int):
    load_library().rism3d_peer_close(int(device), C.c_void_p(ptr))


def rism3d_slab_begin(ctx, tol: float = 0.0):
    _check(ctx, load_library().rism3d_slab_begin(ctx, float(tol)))


def rism3d_slab_phase(ctx, phase: int):
    _check(ctx, load_library().rism3d_slab_phase(ctx, int(phase)))


def rism3d_slab_status(ctx):
    done, n_done, rms = C.c_int(), C.c_int(), C.c_double()
    _check(ctx, load_library().rism3d_slab_status(ctx, C.byref(done), C.byref(n_done), C.byref(rms)))
    return bool(done.value), n_done.value, rms.value


def rism3d_slab_end(ctx):
    n_done, rms = C.c_int(), C.c_double()
    _check(ctx, load_library().rism3d_slab_end(ctx, C.byref(n_done), C.byref(rms)))
    return n_done.value, rms.value


def rism3d_destroy(ctx):
    load_library().rism3d_destroy(ctx)


# ---- convenience object --------------------------------------------------------------------------
class Solver:
    """Owns the workspace tensor and the context; each method is one C-ABI call."""

    def __init__(self, n, spacing, n_sites, closure="KH", pse_order=1, temperature=298.0, mdiis_nvec=5,
                 mdiis_b=0.5, mdiis_restart=10.0, kappa=1.0, r_min=1e-3, origin=None, device=0,
                 accelerator="MDIIS", anderson_s=(0.2, 0.0), mdiis_dynamic_b=None, n_ranks=1, rank=0, stream=None,
                 exportable=False):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("paper_2403_01039_b200 needs a CUDA device (no CPU fallback)")
        load_library()
        # n: points per axis, one number (cube) or (nx, ny, nz); self.n stays the caller's value, self.shape the triple
        self.shape = (int(n),) * 3 if np.isscalar(n) else tuple(int(m) for m in n)
        if len(self.shape) != 3:
            raise ValueError(f"n must be one number or (nx, ny, nz), got {n!r}")
        self.n = int(n) if np.isscalar(n) else self.shape
        self.n_sites, self.spacing = int(n_sites), float(spacing)
        p = Rism3dParams()
        p.nx, p.ny, p.nz = self.shape
        p.spacing = self.spacing
        org = [-(m // 2) * self.spacing for m in self.shape] if origin is None else list(origin)
        p.origin = (C.c_double * 3)(*org)
        p.n_sites = self.n_sites
        p.closure = CLOSURES[closure]
        p.pse_order = int(pse_order)
        p.temperature = float(temperature)
        p.mdiis_nvec = int(mdiis_nvec)
        p.mdiis_b = float(mdiis_b)
        p.mdiis_restart = float(mdiis_restart)
        p.kappa = float(kappa)
        p.r_min = float(r_min)
        p.device = int(device)
        p.accelerator = ACCELERATORS[accelerator]
        p.anderson_s = (C.c_double * 2)(float(anderson_s[0]), float(anderson_s[1]))
        p.mdiis_dynamic_b = 0 if mdiis_dynamic_b is None else 1        # (b_min, b_max) of b = -0.2 log10(rms)
        p.mdiis_b_min, p.mdiis_b_max = (0.0, 0.0) if mdiis_dynamic_b is None else (float(mdiis_dynamic_b[0]), float(mdiis_dynamic_b[1]))
        p.n_ranks, p.rank = int(n_ranks), int(rank)
        self.n_ranks, self.rank = max(1, int(n_ranks)), int(rank)
        self.grid_shape = self.shape                 # the whole grid; self.shape = what this context holds (its slab)
        if self.n_ranks > 1:
            self.shape = (self.shape[0] // self.n_ranks,) + self.shape[1:]
        self.params = p
        nbytes = rism3d_workspace_bytes(p)
        if nbytes == 0:
            raise Rism3dError(-2, "unsupported grid / site count / MDIIS size")
        self.device = torch.device("cuda", device)
        self._raw_workspace = None
        if exportable:
            # an allocation of its own (plain cudaMalloc) that other processes can map: rism3d_peer_export
            self._raw_workspace = rism3d_peer_alloc(device, nbytes)
            self.workspace = None
            self.workspace_ptr, self.workspace_bytes = self._raw_workspace, nbytes
        else:
            self.workspace = torch.empty(nbytes, dtype=torch.uint8, device=self.device)
            self.workspace_ptr, self.workspace_bytes = self.workspace.data_ptr(), nbytes
        # a stream of its own (not the legacy default stream): the library captures its iteration into CUDA graphs
        self.stream = torch.cuda.Stream(self.device) if stream is None else stream
        self.stream.wait_stream(torch.cuda.current_stream(self.device))     # the workspace allocation above
        self.ctx = rism3d_init(p, self.workspace_ptr, nbytes, self.stream.cuda_stream)

    def close(self):
        if getattr(self, "ctx", None) is not None:
            rism3d_destroy(self.ctx)
            self.ctx = None
        if getattr(self, "_raw_workspace", None) is not None:
            rism3d_peer_free(self.device.index, self._raw_workspace)
            self._raw_workspace = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_solvent_chi(self, q, sigma, eps, rho, k0, dk, chi):
        # the C side reads n_sites entries of each array and n_k * n_sites^2 of chi: check before handing pointers over
        q, sigma, eps, rho, chi = _f64(q), _f64(sigma), _f64(eps), _f64(rho), _f64(chi)
        for name, a in (("q", q), ("sigma", sigma), ("eps", eps), ("rho", rho)):
            if a.shape != (self.n_sites,):
                raise ValueError(f"{name} must have shape ({self.n_sites},), got {a.shape}")
        if chi.ndim != 3 or chi.shape[1:] != (self.n_sites, self.n_sites):
            raise ValueError(f"chi must have shape (n_k, {self.n_sites}, {self.n_sites}), got {chi.shape}")
        rism3d_set_solvent_chi(self.ctx, q, sigma, eps, rho, k0, dk, chi)

    def set_solute(self, xyz, q, sigma, eps, rcut=0.0) -> float:
        xyz, q, sigma, eps = _f64(xyz), _f64(np.atleast_1d(q)), _f64(np.atleast_1d(sigma)), _f64(np.atleast_1d(eps))
        n_atoms = len(q)
        xyz = xyz.reshape(0, 3) if xyz.size == 0 else xyz
        if xyz.shape != (n_atoms, 3) or sigma.shape != (n_atoms,) or eps.shape != (n_atoms,):
            raise ValueError(f"solute arrays disagree: xyz {xyz.shape}, q {q.shape}, sigma {sigma.shape}, eps {eps.shape}")
        self.n_atoms = n_atoms
        return rism3d_set_solute(self.ctx, xyz, q, sigma, eps, rcut)

    def gradient(self) -> np.ndarray:
        return rism3d_gradient(self.ctx, self.n_atoms)

    def iterate(self, max_iter, tol=0.0):
        return rism3d_iterate(self.ctx, max_iter, tol)

    def free_energy(self):
        return rism3d_free_energy(self.ctx, self.n_sites)

    def measure_dfma_peak(self) -> float:
        return rism3d_measure_dfma_peak(self.ctx)

    def pressure_correction(self, chi_t: float, pressure: float):
        return rism3d_pressure_correction(self.ctx, chi_t, pressure)

    def phi_ms(self) -> float:
        return rism3d_phi_ms(self.ctx)

    def pmv(self, chi_t: float):
        return rism3d_pmv(self.ctx, chi_t, self.n_sites)

    def get_field(self, which: str, site=None) -> np.ndarray:
        """Host copy: [nx][ny][nz] for one site, or [n_sites][nx][ny][nz] when site is None."""
        sites = range(self.n_sites) if site is None else [site]
        out = np.empty((len(sites),) + self.shape)
        for i, s in enumerate(sites):
            rism3d_get_field(self.ctx, FIELDS[which], s, out[i].ctypes.data, False)
        return out if site is None else out[0]

    def get_field_device(self, which: str, site: int):
        import torch
        out = torch.empty(self.shape, dtype=torch.float64, device=self.device)
        self.stream.wait_stream(torch.cuda.current_stream(self.device))     # the block may have pending uses there
        rism3d_get_field(self.ctx, FIELDS[which], site, out.data_ptr(), True)
        return out

    def set_tau(self, site: int, src):
        import torch
        if isinstance(src, torch.Tensor) and src.is_cuda:
            src = src.contiguous()
            self.stream.wait_stream(torch.cuda.current_stream(self.device))    # src may still be in flight there
            rism3d_set_tau(self.ctx, site, src.data_ptr(), True)
        else:
            a = _f64(src)
            rism3d_set_tau(self.ctx, site, a.ctypes.data, False)

    def rms_history(self) -> np.ndarray:
        return rism3d_get_rms_history(self.ctx)

    def launch_count(self) -> int:
        return rism3d_launch_count(self.ctx)

    def set_profiling(self, enable: bool):
        rism3d_set_profiling(self.ctx, enable)

    def timings(self):
        """-> ({kernel name: mean ms per iteration}, n_iterations) of the profiled iterations"""
        ms, n = rism3d_get_timings(self.ctx)
        return {rism3d_loop_kernel_name(k): (ms[k] / n if n else 0.0) for k in range(N_LOOP_KERNELS)}, n

    @property
    def _padded_sites(self) -> int:
        return 1 if self.n_sites <= 1 else (2 if self.n_sites <= 2 else (4 if self.n_sites <= 4 else 8))

    def fft_forward(self, real_dev):
        """debug: real device tensor [n_sites][nx][ny][nz] -> complex device tensor [nx][ny][nz/2][n_sites]."""
        import torch
        nvp = self._padded_sites                     # the library transforms the padded site count (rism3d.h)
        if nvp != self.n_sites:
            pad = torch.zeros((nvp,) + self.shape, dtype=torch.float64, device=self.device)
            pad[: self.n_sites] = real_dev
            real_dev = pad
        real_dev = real_dev.contiguous()
        nx, ny, nz = self.shape
        out = torch.empty((nx, ny, nz // 2, nvp), dtype=torch.complex128, device=self.device)
        self.stream.wait_stream(torch.cuda.current_stream(self.device))
        rism3d_debug_fft_forward(self.ctx, real_dev.data_ptr(), out.data_ptr())
        return out[..., : self.n_sites]

    def fft_inverse(self, spec_dev):
        import torch
        nvp = self._padded_sites
        if nvp != self.n_sites:
            nx, ny, nz = self.shape
            pad = torch.zeros((nx, ny, nz // 2, nvp), dtype=torch.complex128, device=self.device)
            pad[..., : self.n_sites] = spec_dev
            spec_dev = pad
        spec_dev = spec_dev.contiguous()
        out = torch.empty((nvp,) + self.shape, dtype=torch.float64, device=self.device)
        self.stream.wait_stream(torch.cuda.current_stream(self.device))
        rism3d_debug_fft_inverse(self.ctx, spec_dev.data_ptr(), out.data_ptr())
        return out[: self.n_sites]


# ---- slab-decomposed runs (include/rism3d.h "Slab decomposition") ----------------------------------------------------
class SlabSolver(Solver):
    """One rank of a solve shared by n_ranks GPUs.  Same calls as Solver; fields are this rank's planes
    [nx / n_ranks][ny][nz]; free_energy / pmv / pressure_correction / gradient return the sums over ALL ranks.

    Two ways to run it:
      * one process per GPU under torch.distributed (backend nccl): `group` is the process group (None = the default
        one).  The two transposes are all_to_all_single calls on equal, contiguous blocks that the y passes have
        already laid out per destination, the Gram rows one all_gather -- issued on the solver's stream between the
        phase calls.  `connect_peers(addresses)` switches to peer mode (pointers of every rank's arrays mapped into this
        process, e.g. from torch's symmetric memory): the y passes then store to / load from the other GPUs directly and
        iterate() is a single C call with in-stream barriers.
      * several ranks of one process on one GPU, driven phase by phase by `iterate_in_lockstep` (how the tests check
        the decomposition against the oracle on a single GPU; no rank ever waits for another inside a kernel).
    Only plumbing lives here: every numerical step is a kernel behind rism3d_slab_phase."""

    def __init__(self, n, spacing, n_sites, n_ranks, rank, group=None, **kw):
        super().__init__(n, spacing, n_sites, n_ranks=n_ranks, rank=rank, **kw)
        import torch
        self.group = group
        loc = rism3d_slab_local(self.ctx)
        self.local = loc
        base = self.workspace_ptr
        self.K = self.stage = self.gram = None
        if self.workspace is not None:                  # (an exportable workspace is for peer mode: nothing is staged)
            def view(addr, nbytes):
                return self.workspace[addr - base: addr - base + nbytes].view(torch.float64)

            nb = loc["block_bytes"] * self.n_ranks
            self.K = view(loc["K"], nb)                 # [n_ranks][block]: block s came from rank s
            self.stage = view(loc["stage"], nb)         # [n_ranks][block]: block d goes to rank d / came back from it
            self.gram = view(loc["gram"], loc["gram_row_bytes"] * self.n_ranks)
        self.peer_mode = False
        self._opened = []

    # -- phase calls ---------------------------------------------------------------------------------------------
    def begin(self, tol=0.0):
        rism3d_slab_begin(self.ctx, tol)

    def phase(self, k):
        rism3d_slab_phase(self.ctx, k)

    def status(self):
        return rism3d_slab_status(self.ctx)

    def end(self):
        return rism3d_slab_end(self.ctx)

    def connect_peers(self, d_K, d_gram, d_flags):
        rism3d_slab_set_peers(self.ctx, d_K, d_gram, d_flags)
        self.peer_mode = True

    def set_peer_timeout(self, seconds: float):
        rism3d_slab_set_peer_timeout(self.ctx, seconds)

    def connect_peers_ipc(self):
        """Peer mode across processes (one GPU each, one node): every rank exports its workspace (created with
        exportable=True), the handles travel through the process group, every rank maps the others' workspaces (CUDA
        IPC; the arrays sit at the same offsets everywhere) and hands the addresses to rism3d_slab_set_peers."""
        import torch.distributed as dist
        if self._raw_workspace is None:
            raise RuntimeError("connect_peers_ipc needs SlabSolver(..., exportable=True)")
        handles = [None] * self.n_ranks
        dist.all_gather_object(handles, rism3d_peer_export(self.device.index, self._raw_workspace), group=self.group)
        off = {k: self.local[k] - self.workspace_ptr for k in ("K", "gram", "flags")}
        bases = []
        for r in range(self.n_ranks):
            if r == self.rank:
                bases.append(self.workspace_ptr)
            else:
                bases.append(rism3d_peer_open(self.device.index, handles[r]))
                self._opened.append(bases[-1])
        self.connect_peers([b + off["K"] for b in bases], [b + off["gram"] for b in bases], [b + off["flags"] for b in bases])
        dist.barrier(group=self.group)

    def iterate_host_ordered(self, max_iter, tol=0.0, check_every=8):
        """Peer mode with the ranks kept in step by the HOST (stream synchronise + process-group barrier where the
        phases meet) instead of the in-stream barrier kernel: for ranks whose kernels cannot be relied on to run at the
        same time (several ranks time-slicing one GPU, as in the tests)."""
        import torch.distributed as dist
        if not self.peer_mode:
            raise RuntimeError("iterate_host_ordered is for peer mode (connect_peers / connect_peers_ipc)")

        def meet():
            self.stream.synchronize()
            dist.barrier(group=self.group)

        self.begin(tol)
        for it in range(max_iter):
            self.phase(0); meet()
            self.phase(1); meet()
            self.phase(2); meet()
            self.phase(3)
            if tol > 0.0 and (it + 1) % check_every == 0 and self.status()[0]:
                break
        out = self.end()
        meet()
        return out

    def close(self):
        for ptr in getattr(self, "_opened", []):
            rism3d_peer_close(self.device.index, ptr)
        self._opened = []
        super().close()

    # -- one process per GPU -------------------------------------------------------------------------------------
    def _device_collectives(self) -> bool:
        """True when the process group moves device tensors itself (nccl); any other backend (gloo, in the CPU-side
        tests and on boxes without NVLink) gets the blocks through host memory."""
        import torch.distributed as dist
        return dist.get_backend(self.group) == "nccl"

    def _all_to_all(self, dst, src):
        import torch
        import torch.distributed as dist
        if self._device_collectives():
            dist.all_to_all_single(dst, src, group=self.group)
        else:
            h_src = src.cpu()                            # synchronises the solver's stream (the current one here)
            h_dst = torch.empty_like(h_src)
            dist.all_to_all_single(h_dst, h_src, group=self.group)
            dst.copy_(h_dst)

    def _all_gather_rows(self):
        import torch
        import torch.distributed as dist
        row = self.gram.numel() // self.n_ranks
        mine = self.gram[self.rank * row:(self.rank + 1) * row]
        if self._device_collectives():
            dist.all_gather_into_tensor(self.gram, mine, group=self.group)
        else:
            h = torch.empty(self.gram.numel(), dtype=torch.float64)
            dist.all_gather_into_tensor(h, mine.cpu(), group=self.group)
            self.gram.copy_(h)

    def iterate(self, max_iter, tol=0.0, check_every=8):
        if self.peer_mode:
            return rism3d_iterate(self.ctx, max_iter, tol)
        import torch
        self.begin(tol)
        with torch.cuda.stream(self.stream):
            for it in range(max_iter):
                self.phase(0)
                self._all_to_all(self.K, self.stage)                                  # forward transpose
                self.phase(1)
                self._all_to_all(self.stage, self.K)                                  # backward transpose
                self.phase(2)
                self._all_gather_rows()
                self.phase(3)
                if tol > 0.0 and (it + 1) % check_every == 0 and self.status()[0]:
                    break
        return self.end()

    def _sum_over_ranks(self, values):
        """all-gather the ranks' shares (data movement), add them in rank order inside the library (rism3d_slab_combine)"""
        import torch
        import torch.distributed as dist
        t = torch.as_tensor(np.ascontiguousarray(np.asarray(values, dtype=np.float64).reshape(-1)))
        if self._device_collectives():
            t = t.to(self.device)
        rows = torch.empty(self.n_ranks * t.numel(), dtype=torch.float64, device=t.device)     # flat: rank r's share at r * n
        dist.all_gather_into_tensor(rows, t, group=self.group)
        return rism3d_slab_combine(rows.cpu().numpy().reshape(self.n_ranks, t.numel())).reshape(np.shape(values))

    def free_energy(self):
        mu, site = rism3d_free_energy(self.ctx, self.n_sites)
        tot = self._sum_over_ranks(np.concatenate([[mu], site]))
        return float(tot[0]), tot[1:]

    def pmv(self, chi_t: float):
        v, c_int = rism3d_pmv(self.ctx, chi_t, self.n_sites)
        tot = self._sum_over_ranks(np.concatenate([[v], c_int]))
        return float(tot[0]), tot[1:]

    def pressure_correction(self, chi_t: float, pressure: float):
        # every rank's call returns its share of -P V (Eq. 21) and of V: both are sums over the slabs
        pc, v = rism3d_pressure_correction(self.ctx, chi_t, pressure)
        tot = self._sum_over_ranks(np.array([pc, v]))
        return float(tot[0]), float(tot[1])

    def gradient(self) -> np.ndarray:
        return self._sum_over_ranks(rism3d_gradient(self.ctx, self.n_atoms))


def iterate_in_lockstep(ranks, max_iter, tol=0.0):
    """Drive all ranks of a slab run that live in ONE process on ONE GPU (SlabSolver objects created with the same
    `stream`), phase by phase.  Staged mode: the blocks move by device copies that stand in for the all-to-all; peer
    mode (after connect_peers with each other's addresses): nothing to move.  -> (n_done, rms) of rank 0."""
    import torch
    P = len(ranks)
    stream = ranks[0].stream
    assert all(r.stream is stream for r in ranks), "lockstep ranks share one stream"
    peer = ranks[0].peer_mode
    blk = ranks[0].local["block_bytes"] // 8
    row = ranks[0].local["gram_row_bytes"] // 8
    for r in ranks:
        r.begin(tol)
    with torch.cuda.stream(stream):
        for it in range(max_iter):
            for r in ranks:
                r.phase(0)
            if not peer:
                for d in range(P):
                    for s in range(P):
                        ranks[d].K[s * blk:(s + 1) * blk].copy_(ranks[s].stage[d * blk:(d + 1) * blk])
            for r in ranks:
                r.phase(1)
            if not peer:
                for d in range(P):
                    for s in range(P):
                        ranks[d].stage[s * blk:(s + 1) * blk].copy_(ranks[s].K[d * blk:(d + 1) * blk])
            for r in ranks:
                r.phase(2)
            if not peer:
                for d in range(P):
                    for s in range(P):
                        if s != d:
                            ranks[d].gram[s * row:(s + 1) * row].copy_(ranks[s].gram[s * row:(s + 1) * row])
            for r in ranks:
                r.phase(3)
            if tol > 0.0 and (it + 1) % 8 == 0 and ranks[0].status()[0]:
                break
    out = [r.end() for r in ranks]
    return out[0]


# ---- the 1D solvent solve (include/rism1d.h) ---------------------------------------------------------------------------
def _check1(ctx, status: int):
    if status != 0:
        lib = load_library()
        msg = lib.rism1d_last_error(ctx).decode() if ctx else ""
        raise Rism3dError(status, msg or lib.rism3d_status_string(status).decode())


def rism1d_workspace_bytes(params: Rism1dParams) -> int:
    return int(load_library().rism1d_workspace_bytes(C.byref(params)))


def rism1d_init(params: Rism1dParams, d_workspace: int, nbytes: int, cuda_stream: int):
    ctx = C.c_void_p()
    st = load_library().rism1d_init(C.byref(ctx), C.byref(params), C.c_void_p(d_workspace), nbytes, C.c_void_p(cuda_stream))
    if st != 0:
        raise Rism3dError(st, rism3d_status_string(st))
    return ctx


def rism1d_set_solvent(ctx, q, sigma, eps, rho_site, species, bond):
    q, sigma, eps, rho_site, bond = _f64(q), _f64(sigma), _f64(eps), _f64(rho_site), _f64(bond)
    species = np.ascontiguousarray(np.asarray(species, dtype=np.int32))
    _check1(ctx, load_library().rism1d_set_solvent(ctx, _dptr(q), _dptr(sigma), _dptr(eps), _dptr(rho_site),
                                                   species.ctypes.data_as(C.POINTER(C.c_int)), _dptr(bond)))


def rism1d_solve(ctx, charge_scale: float, max_iter: int, tol: float):
    n_done, rms = C.c_int(), C.c_double()
    _check1(ctx, load_library().rism1d_solve(ctx, float(charge_scale), int(max_iter), float(tol), C.byref(n_done), C.byref(rms)))
    return n_done.value, rms.value


def rism1d_get_pair(ctx, which: int, n_sites: int, n_points: int) -> np.ndarray:
    out = np.empty((n_sites, n_sites, n_points - 1))
    _check1(ctx, load_library().rism1d_get_pair(ctx, int(which), _dptr(out)))
    return out


def rism1d_get_chi(ctx, n_sites: int, n_points: int) -> np.ndarray:
    out = np.empty((n_points - 1, n_sites, n_sites))
    _check1(ctx, load_library().rism1d_get_chi(ctx, _dptr(out)))
    return out


def rism1d_get_chi_types(ctx, site_type, n_points: int) -> np.ndarray:
    st = np.ascontiguousarray(np.asarray(site_type, dtype=np.int32))
    n_types = int(st.max()) + 1
    out = np.empty((n_points - 1, n_types, n_types))
    _check1(ctx, load_library().rism1d_get_chi_types(ctx, n_types, st.ctypes.data_as(C.POINTER(C.c_int)), _dptr(out)))
    return out


def rism1d_thermo(ctx, n_sites: int):
    chi_t, pr = C.c_double(), C.c_double()
    c0 = np.empty((n_sites, n_sites))
    _check1(ctx, load_library().rism1d_thermo(ctx, C.byref(chi_t), C.byref(pr), _dptr(c0)))
    return chi_t.value, pr.value, c0


def rism1d_launch_count(ctx) -> int:
    return int(load_library().rism1d_launch_count(ctx))


def rism1d_last_error(ctx) -> str:
    return load_library().rism1d_last_error(ctx).decode()


def rism1d_destroy(ctx):
    load_library().rism1d_destroy(ctx)


class Solver1d:
    """Solvent-solvent 1D-RISM on the GPU: owns the workspace and the context; each method is one C-ABI call (the
    charge ramp is a loop of solve calls).  Produces chi for rism3d_set_solvent_chi, chi_T and P."""

    PAIRS = {"G": 0, "TAU": 1, "C_SR": 2}

    def __init__(self, n_sites, n_points=16384, dr=0.025, temperature=298.0, kappa=1.0, closure="KH", pse_order=1,
                 mdiis_nvec=10, mdiis_b=0.5, mdiis_restart=10.0, device=0):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("paper_2403_01039_b200 needs a CUDA device (no CPU fallback)")
        load_library()
        p = Rism1dParams()
        p.n_sites, p.n_points, p.dr, p.temperature, p.kappa = int(n_sites), int(n_points), float(dr), float(temperature), float(kappa)
        p.closure, p.pse_order = CLOSURES[closure], int(pse_order)
        p.mdiis_nvec, p.mdiis_b, p.mdiis_restart, p.device = int(mdiis_nvec), float(mdiis_b), float(mdiis_restart), int(device)
        self.params, self.n_sites, self.n_points, self.dr = p, int(n_sites), int(n_points), float(dr)
        nbytes = rism1d_workspace_bytes(p)
        if nbytes == 0:
            raise Rism3dError(-2, "unsupported site count / radial grid / MDIIS size")
        self.device = torch.device("cuda", device)
        self.workspace = torch.empty(nbytes, dtype=torch.uint8, device=self.device)
        self.stream = torch.cuda.Stream(self.device)
        self.stream.wait_stream(torch.cuda.current_stream(self.device))
        self.ctx = rism1d_init(p, self.workspace.data_ptr(), nbytes, self.stream.cuda_stream)

    @property
    def k(self) -> np.ndarray:
        return np.arange(1, self.n_points) * (np.pi / (self.n_points * self.dr))

    @property
    def r(self) -> np.ndarray:
        return np.arange(1, self.n_points) * self.dr

    def close(self):
        if getattr(self, "ctx", None) is not None:
            rism1d_destroy(self.ctx)
            self.ctx = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_solvent(self, q, sigma, eps, rho_site, species, bond):
        n = self.n_sites
        for name, a in (("q", q), ("sigma", sigma), ("eps", eps), ("rho_site", rho_site), ("species", species)):
            if np.shape(a) != (n,):
                raise ValueError(f"{name} must have shape ({n},), got {np.shape(a)}")
        if np.shape(bond) != (n, n):
            raise ValueError(f"bond must have shape ({n}, {n}), got {np.shape(bond)}")
        rism1d_set_solvent(self.ctx, q, sigma, eps, rho_site, species, bond)

    def solve(self, charge_scale=1.0, max_iter=5000, tol=1e-10):
        return rism1d_solve(self.ctx, charge_scale, max_iter, tol)

    def pair(self, which="G") -> np.ndarray:
        return rism1d_get_pair(self.ctx, self.PAIRS[which], self.n_sites, self.n_points)

    def chi(self) -> np.ndarray:
        return rism1d_get_chi(self.ctx, self.n_sites, self.n_points)

    def chi_types(self, site_type) -> np.ndarray:
        return rism1d_get_chi_types(self.ctx, site_type, self.n_points)

    def thermo(self):
        """-> (chi_T [A^3 mol/kcal], P [kcal/(mol A^3)], int c_sr,ab dr [n][n])"""
        return rism1d_thermo(self.ctx, self.n_sites)

    def launch_count(self) -> int:
        return rism1d_launch_count(self.ctx)
