"""Shared test helpers (inputs only, no method arithmetic beyond building synthetic chi tables)."""
import numpy as np


def synthetic_chi(n_v, rho, n_k=600, dk=0.03, k0=0.03, seed=0, amp=0.8):
    """A smooth, physically shaped but made-up susceptibility: chi_{g'g}(k) = delta + rho_{g'} A_{g'g} exp(-(k/2)^2)
    with A symmetric (so that mult-weighted chi is symmetric like a real one)."""
    rng = np.random.default_rng(seed)
    A = rng.uniform(-1.0, 1.0, (n_v, n_v))
    A = 0.5 * (A + A.T) * amp / np.max(rho)
    k = k0 + dk * np.arange(n_k)
    chi = np.eye(n_v)[None] + (np.asarray(rho)[None, :, None] * A[None]) * np.exp(-(k / 2.0) ** 2)[:, None, None]
    return k0, dk, chi


def identity_chi(n_v, n_k=600, dk=0.03, k0=0.03):
    return k0, dk, np.tile(np.eye(n_v)[None], (n_k, 1, 1))
