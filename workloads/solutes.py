"""Seeded synthetic solutes, one recipe per BASELINE.json config.

Every generator uses `numpy.random.default_rng(seed)` (PCG64) and returns a `Solute` whose
coordinates are shifted so that the centroid sits at the coordinate origin (C1 keeps its single
atom exactly at 0).  Units: Angstrom, e, kcal/mol.
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np

MIN_SEP = 1.2     # A, minimum atom-atom separation in every multi-atom recipe
BOND_STEP = 3.8   # A, chain step of the protein-like recipes


@dataclass
class Solute:
    name: str
    xyz: np.ndarray      # [n][3]
    q: np.ndarray        # [n]
    sigma: np.ndarray    # [n]
    eps: np.ndarray      # [n]

    @property
    def n_atoms(self) -> int:
        return len(self.q)


def _unit_vectors(rng, n):
    v = rng.standard_normal((n, 3))
    return v / np.linalg.norm(v, axis=1, keepdims=True)


def _lj(rng, n):
    sigma = rng.uniform(2.5, 3.8, n)
    eps = rng.uniform(0.05, 0.2, n)
    return sigma, eps


def _charges(rng, n, width, total):
    q = rng.normal(0.0, width, n)
    q += (total - q.sum()) / n
    return q


def _sphere_cloud(rng, n, radius, placed=None):
    """Sequential rejection sampling, uniform in a sphere, >= MIN_SEP from all accepted atoms."""
    pts = np.empty((n, 3))
    k = 0
    while k < n:
        p = _unit_vectors(rng, 1)[0] * radius * rng.uniform() ** (1.0 / 3.0)
        if k and np.min(np.sum((pts[:k] - p) ** 2, axis=1)) < MIN_SEP ** 2:
            continue
        pts[k] = p
        k += 1
    return pts


def _confined_chain(rng, n, radius, centre, others=None):
    """Random-walk chain with BOND_STEP steps, confined to a sphere, self- and cross-avoiding.

    Each step is redrawn up to 1000 times if it leaves the sphere or comes closer than MIN_SEP to
    an earlier atom (of this chain or of `others`); on failure the walk backs up 10 atoms.
    """
    pts = np.empty((n, 3))
    pts[0] = centre
    k = 1
    while k < n:
        ok = False
        for _ in range(1000):
            p = pts[k - 1] + BOND_STEP * _unit_vectors(rng, 1)[0]
            if np.sum((p - centre) ** 2) > radius ** 2:
                continue
            if np.min(np.sum((pts[:k] - p) ** 2, axis=1)) < MIN_SEP ** 2:
                continue
            if others is not None and len(others) and \
                    np.min(np.sum((others - p) ** 2, axis=1)) < MIN_SEP ** 2:
                continue
            ok = True
            break
        if ok:
            pts[k] = p
            k += 1
        else:
            k = max(1, k - 10)
    return pts


def make_c1() -> Solute:
    """Single Na+ ion at the origin (BASELINE.json configs[0])."""
    return Solute("C1_na_ion", np.zeros((1, 3)), np.array([1.0]), np.array([2.35]), np.array([0.13]))


def make_c2(seed: int = 2) -> Solute:
    rng = np.random.default_rng(seed)
    n = 20
    xyz = _sphere_cloud(rng, n, 6.0)
    q = _charges(rng, n, 0.3, 0.0)
    sigma, eps = _lj(rng, n)
    xyz -= xyz.mean(axis=0)
    return Solute("C2_organic20", xyz, q, sigma, eps)


def make_c3(seed: int = 3) -> Solute:
    rng = np.random.default_rng(seed)
    n = 500
    xyz = _sphere_cloud(rng, n, 18.0)
    q = _charges(rng, n, 0.3, 3.0)
    sigma, eps = _lj(rng, n)
    xyz -= xyz.mean(axis=0)
    return Solute("C3_cluster500", xyz, q, sigma, eps)


def make_c4(seed: int = 4, n: int = 2000) -> Solute:
    rng = np.random.default_rng(seed)
    xyz = _confined_chain(rng, n, 25.0, np.zeros(3))
    q = _charges(rng, n, 0.4, 8.0)
    sigma, eps = _lj(rng, n)
    xyz -= xyz.mean(axis=0)
    return Solute("C4_chain2000", xyz, q, sigma, eps)


def make_c5(seed: int = 5, n_chains: int = 10, n_per_chain: int = 2000) -> Solute:
    rng = np.random.default_rng(seed)
    centres = []
    while len(centres) < n_chains:
        c = _unit_vectors(rng, 1)[0] * 55.0 * rng.uniform() ** (1.0 / 3.0)
        if all(np.linalg.norm(c - d) >= 40.0 for d in centres):
            centres.append(c)
    chunks, qs = [], []
    placed = np.empty((0, 3))
    for ci, c in enumerate(centres):
        crng = np.random.default_rng(seed + 1 + ci)
        # a neighbouring sphere may touch this one: test against every atom placed so far
        pts = _confined_chain(crng, n_per_chain, 25.0, c, others=placed)
        placed = np.concatenate([placed, pts])
        chunks.append(pts)
        qs.append(crng.normal(0.0, 0.4, n_per_chain))
    xyz = np.concatenate(chunks)
    q = np.concatenate(qs)
    q += (-20.0 - q.sum()) / len(q)
    n = len(q)
    sigma, eps = _lj(rng, n)
    xyz -= xyz.mean(axis=0)
    return Solute("C5_multidomain20000", xyz, q, sigma, eps)


_MAKERS = {"C1": make_c1, "C2": make_c2, "C3": make_c3, "C4": make_c4, "C5": make_c5}
_CACHE: dict = {}


def make_solute(config_name: str) -> Solute:
    if config_name not in _CACHE:
        _CACHE[config_name] = _MAKERS[config_name]()
    return _CACHE[config_name]
