"""Solvent site parameters (inputs only; BASELINE.json `configs`).

Units: charge e, sigma Angstrom, eps kcal/mol, density Angstrom^-3.

Two views of the same solvent are kept:
  * full-site view (one entry per atom of each species; used by the 1D solvent solve),
  * type view (identical atoms of a species merged: water -> O, H; used by the 3D path), where
    rho_type = multiplicity x species number density.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

N_AVOGADRO = 6.02214076e23
RHO_WATER = 0.0334          # molecules / A^3 (BASELINE.json configs[0])
L_OH = 1.0                  # A, "SPC/E-like" geometry
L_HH = 1.63299              # A (109.47 deg)


@dataclass
class Solvent:
    name: str
    # ---- type view (what the 3D path consumes) ----
    type_names: list
    q: np.ndarray            # [n_v]
    sigma: np.ndarray        # [n_v]
    eps: np.ndarray          # [n_v]
    rho: np.ndarray          # [n_v]  type density = mult * species density
    mult: np.ndarray         # [n_v]  multiplicity of the type inside its species
    # ---- full-site view (what the 1D solvent solve consumes) ----
    site_type: np.ndarray    # [n_s] index into the type arrays
    site_species: np.ndarray  # [n_s] species index
    species_rho: np.ndarray  # [n_species]
    bond: np.ndarray         # [n_s][n_s] intramolecular distance (0 on the diagonal / across species)
    meta: dict = field(default_factory=dict)

    @property
    def n_v(self) -> int:
        return len(self.type_names)

    @property
    def n_s(self) -> int:
        return len(self.site_type)


def molar_to_number_density(conc_molar: float) -> float:
    """mol/L -> particles / A^3  (1 L = 1e27 A^3)."""
    return conc_molar * N_AVOGADRO * 1e-27


def water() -> Solvent:
    bond = np.zeros((3, 3))
    bond[0, 1] = bond[1, 0] = L_OH
    bond[0, 2] = bond[2, 0] = L_OH
    bond[1, 2] = bond[2, 1] = L_HH
    return Solvent(
        name="water",
        type_names=["O", "H"],
        q=np.array([-0.8476, 0.4238]),
        sigma=np.array([3.166, 1.0]),
        eps=np.array([0.1553, 0.046]),
        rho=np.array([RHO_WATER, 2 * RHO_WATER]),
        mult=np.array([1, 2]),
        site_type=np.array([0, 1, 1]),
        site_species=np.array([0, 0, 0]),
        species_rho=np.array([RHO_WATER]),
        bond=bond,
    )


def water_nacl(conc_molar: float) -> Solvent:
    """Water + NaCl at `conc_molar` mol/L: 4 site types O, H, Na+, Cl- (BASELINE.json configs[2..4])."""
    w = water()
    rho_ion = molar_to_number_density(conc_molar)
    bond = np.zeros((5, 5))
    bond[:3, :3] = w.bond
    return Solvent(
        name=f"water_nacl_{conc_molar:g}M",
        type_names=["O", "H", "Na+", "Cl-"],
        q=np.array([-0.8476, 0.4238, 1.0, -1.0]),
        sigma=np.array([3.166, 1.0, 2.35, 4.4]),
        eps=np.array([0.1553, 0.046, 0.13, 0.1]),
        rho=np.array([RHO_WATER, 2 * RHO_WATER, rho_ion, rho_ion]),
        mult=np.array([1, 2, 1, 1]),
        site_type=np.array([0, 1, 1, 2, 3]),
        site_species=np.array([0, 0, 0, 1, 2]),
        species_rho=np.array([RHO_WATER, rho_ion, rho_ion]),
        bond=bond,
        meta={"conc_molar": conc_molar},
    )


def solvent_by_name(name: str) -> Solvent:
    if name == "water":
        return water()
    if name.startswith("water_nacl_") and name.endswith("M"):
        return water_nacl(float(name[len("water_nacl_"):-1]))
    raise KeyError(name)
