"""Seeded synthetic input generators shared by the oracle tests and the GPU parity tests.

Holds NONE of the method's arithmetic (no kicks, hops, plaquettes, windings): only numpy random
numbers shaped into the canonical state layout (20, nz, ny, nx), float64:
  0 phi_re 1 phi_im 2 Pi_re 3 Pi_im 4 psi_re 5 psi_im 6 Psi_re 7 Psi_im
  8..10 thetaA_xyz 11..13 E_xyz 14..16 thetaB_xyz 17..19 H_xyz
"""
from __future__ import annotations

import numpy as np

POS = [0, 1, 4, 5, 8, 9, 10, 14, 15, 16]
MOM = [2, 3, 6, 7, 11, 12, 13, 17, 18, 19]
GROUPS = {
    "phi": [0, 1], "Pi": [2, 3], "psi": [4, 5], "Psi": [6, 7],
    "thetaA": [8, 9, 10], "E": [11, 12, 13], "thetaB": [14, 15, 16], "H": [17, 18, 19],
}


def _smooth(rng, shape, passes=2):
    """White noise averaged with periodic nearest neighbours a few times (just a smooth random field)."""
    a = rng.standard_normal(shape)
    for _ in range(passes):
        for ax in range(a.ndim):
            a = (np.roll(a, 1, ax) + 2 * a + np.roll(a, -1, ax)) / 4
    return a / np.std(a)


def random_state(shape, seed, amp_mom=0.3, amp_theta=0.8, smooth=True, modulus_jitter=0.2):
    """A generic state exercising every term: |phi|,|psi| ~ 1 with jitter, smooth random phases,
    non-zero links and momenta.  shape = (nz, ny, nx).  NOT Gauss-law satisfying (by design)."""
    rng = np.random.default_rng(seed)
    mk = (lambda: _smooth(rng, shape)) if smooth else (lambda: rng.standard_normal(shape))
    s = np.zeros((20,) + tuple(shape))
    for base in (0, 4):
        phase = np.pi * mk()
        mod = 1.0 + modulus_jitter * mk()
        s[base] = mod * np.cos(phase)
        s[base + 1] = mod * np.sin(phase)
    for c in (8, 9, 10, 14, 15, 16):
        s[c] = amp_theta * mk()
    for c in MOM:
        s[c] = amp_mom * mk()
    return s


def to_f32_exact(state):
    """Round to float32 and back so that oracle (fp64) and GPU (fp32) start from IDENTICAL numbers."""
    return state.astype(np.float32).astype(np.float64)


def vortex_pair_phase(shape, centers, charges):
    """Sum of 2-D polar angles around (x0, y0) lines running along z (no lattice arithmetic of the method;
    just atan2 geometry with nearest-image wrapping so the phase is single valued away from the lines)."""
    nz, ny, nx = shape
    y, x = np.meshgrid(np.arange(ny), np.arange(nx), indexing="ij")
    ph = np.zeros((ny, nx))
    for (x0, y0), q in zip(centers, charges):
        ph += q * np.arctan2(y - y0, x - x0)
    return np.broadcast_to(ph, shape).copy()
