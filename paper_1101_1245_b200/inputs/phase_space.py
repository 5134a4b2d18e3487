"""Seeded synthetic phase spaces (input data only).

The paper lists "phase space and spectrum files" as future work; no phase-space
file is in the container, so this generator stands in for the output of a treatment-head
simulation scored on the plane z = 0: photons of a thick-target bremsstrahlung spectrum diverging
from a point focus above the phantom, with a small share of contaminant electrons.  A record is
8 float32 numbers {x, y, z, u, v, w, E, type}; type 0.0 photon, 1.0 electron
(include/gpumcd.h, gpumcd_source.phsp).
"""
from __future__ import annotations

import numpy as np

from .spectra import thick_target_spectrum


def synthetic_phase_space(n: int, seed: int, cx: float, cy: float, wx: float, wy: float, *,
                          focus_cm: float = 100.0, e0: float = 6.0, electron_share: float = 0.05,
                          e_lo: float = 0.25) -> np.ndarray:
    """float32[n, 8]: positions uniform over the wx x wy field centred (cx, cy) on z = 0, directions
    along the ray from a focus `focus_cm` above the field centre, photon energies from the
    thick-target shape up to e0, electron energies uniform on [e_lo, e0 / 2]."""
    rng = np.random.default_rng(seed)
    x = cx + (rng.random(n) - 0.5) * wx
    y = cy + (rng.random(n) - 0.5) * wy
    d = np.stack([x - cx, y - cy, np.full(n, focus_cm)], axis=1)
    d /= np.linalg.norm(d, axis=1, keepdims=True)
    edges, w = thick_target_spectrum(e0, e_lo, 256)
    cdf = np.cumsum(w.astype(np.float64))
    j = np.searchsorted(cdf, rng.random(n) * cdf[-1], side="right").clip(0, w.size - 1)
    e_ph = edges[j] + rng.random(n) * (edges[j + 1] - edges[j])
    is_e = rng.random(n) < electron_share
    e_el = e_lo + rng.random(n) * (0.5 * e0 - e_lo)
    rec = np.empty((n, 8), np.float32)
    rec[:, 0], rec[:, 1], rec[:, 2] = x, y, 0.0
    rec[:, 3:6] = d
    rec[:, 6] = np.where(is_e, e_el, e_ph)
    rec[:, 7] = is_e
    return rec
