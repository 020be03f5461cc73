"""CPU oracle for the 3D-RISM hot path of arxiv 2403.01039 (RISMiCal) -- TEST INFRASTRUCTURE ONLY.

Plain, slow, double-precision numpy restatement of what the path computes, written from
/root/reference/PAPER.md (cited as PAPER.md:<line>) with the readings listed in DESIGN.md.
It shares no code with the CUDA path (`paper_2403_01039_b200/`), imports nothing from it, and is
imported only by `tests/`, `__graft_entry__.smoke()` and `bench.py`'s cpu_baseline / reference leg.

Modules
  rism3d.py           O-3D: potential, long-range split, closure, shifted DFT, 3D-RISM loop, MDIIS, SFE
  rism1d.py           O-1D: 1D XRISM solvent solve -> chi ; 1D solute-solvent solve (spherical-ion pin)
  make_chi_tables.py  script: writes workloads/chi/*.npz by calling rism1d only

Parity pins: every function here is pinned by `tests/test_oracle_*.py` (brute-force DFT, closed
forms, invariants, textbook special cases); the paper's printed SFE/PMV values need
the paper's protein data set, which is not available, and stay "parity unpinned".
"""
