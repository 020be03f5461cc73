"""B200-native 3D-RISM solver core (arxiv 2403.01039, RISMiCal): Python binding of librism3d.so.

Everything numerical runs in the hand-written sm_100a kernels behind the C ABI of include/rism3d.h;
this package only marshals arguments (ctypes) and uses PyTorch for device memory and streams.
There is no CPU fallback: importing works anywhere, but creating a solver without the built library
or without a CUDA device raises.
"""
from .binding import (  # noqa: F401
    ACCELERATORS, CLOSURES, FIELDS, Rism3dError, Rism3dParams, Solver, library_path, load_library,
    rism3d_workspace_bytes, rism3d_init, rism3d_set_solvent_chi, rism3d_set_solute, rism3d_iterate,
    rism3d_free_energy, rism3d_pmv, rism3d_pressure_correction, rism3d_gradient, rism3d_get_field, rism3d_set_tau, rism3d_get_rms_history, rism3d_launch_count, rism3d_phi_ms, rism3d_measure_dfma_peak,
    rism3d_set_profiling, rism3d_get_timings, rism3d_loop_kernel_name, N_LOOP_KERNELS,
    rism3d_debug_fft_forward, rism3d_debug_fft_inverse, rism3d_last_error, rism3d_status_string,
    rism3d_destroy, EXPORTED_SYMBOLS, Rism3dSlabInfo, rism3d_slab_plan, rism3d_slab_local, rism3d_slab_set_peers,
    rism3d_slab_begin, rism3d_slab_phase, rism3d_slab_set_peer_timeout, rism3d_slab_combine, rism3d_debug_peer_barrier_selftest, rism3d_slab_status, rism3d_slab_end, SlabSolver, iterate_in_lockstep,
    rism3d_peer_alloc, rism3d_peer_free, rism3d_peer_export, rism3d_peer_open, rism3d_peer_close,
    EXPORTED_SYMBOLS_1D, Rism1dParams, Solver1d, rism1d_workspace_bytes, rism1d_init, rism1d_set_solvent, rism1d_solve,
    rism1d_get_pair, rism1d_get_chi, rism1d_get_chi_types, rism1d_thermo, rism1d_launch_count, rism1d_last_error,
    rism1d_destroy,
    EXPORTED_SYMBOLS_NOALLOC, NOALLOC_MAX_SITES, NOALLOC_MAX_POINTS, NOALLOC_SCRATCH_BYTES, rism3d_noalloc_free_energy,
)
