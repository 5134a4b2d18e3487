"""Seeded analytic source spectra (input data only).

Config 5 of BASELINE.json asks for a "polyenergetic 18 MV photon beam (spectrum
from a seeded analytic thick-target bremsstrahlung shape, 0.1-18 MeV)".  The
paper has no spectrum source (future work), so the shape is a
choice of this build: p(E) ~ (E0/E - 1) exp(-1/E), the Kramers thick-target
form times a low-energy filtration roll-off.  The shape is deterministic; the
"seed" of the config only enters through the run seed.
"""
from __future__ import annotations

import numpy as np


def thick_target_spectrum(e0: float = 18.0, e_lo: float = 0.1, n_bins: int = 512):
    """Return (edges float32[n_bins+1], weights float32[n_bins]); weights = p(bin centre)."""
    edges = np.linspace(e_lo, e0, n_bins + 1)
    c = 0.5 * (edges[:-1] + edges[1:])
    w = (e0 / c - 1.0) * np.exp(-1.0 / c)
    w = w / w.sum()
    return edges.astype(np.float32), w.astype(np.float32)
