"""Synthetic material definitions (input data only).

These compositions *define* the synthetic materials of the five BASELINE.json
configs; they are standard-looking tissue recipes, not
certified data.  The paper itself only names the media (water, lung, soft
tissue, bone: PAPER.md L233-266) and takes its data from EGSnrc files that are
not available here.

Nothing in this module is transport arithmetic: it is consumed by
``tables.py`` to produce the cross-section / stopping-power tables that are
handed, as plain arrays, to both the CUDA library and the CPU oracle.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Dict, Tuple

# element symbol -> (Z, A [g/mol])
ELEMENTS: Dict[str, Tuple[int, float]] = {
    "H": (1, 1.008),
    "C": (6, 12.011),
    "N": (7, 14.007),
    "O": (8, 15.999),
    "Na": (11, 22.990),
    "Mg": (12, 24.305),
    "P": (15, 30.974),
    "S": (16, 32.06),
    "Cl": (17, 35.45),
    "Ar": (18, 39.948),
    "K": (19, 39.098),
    "Ca": (20, 40.078),
}


@dataclass(frozen=True)
class Material:
    name: str
    weights: Dict[str, float]          # elemental weight fractions, sum to 1
    I_eV: float                        # mean excitation energy
    density: float                     # nominal density, g/cm^3
    gas: bool = False                  # selects the gas branch of the density-effect recipe
    sternheimer: Tuple[float, ...] = field(default=())  # (Cbar, x0, x1, a, m) if fitted values exist

    def za_ratio(self) -> float:
        """<Z/A> = sum_i w_i Z_i / A_i  (mol electrons per gram)."""
        return sum(w * ELEMENTS[e][0] / ELEMENTS[e][1] for e, w in self.weights.items())


WATER = Material(
    "water", {"H": 0.1119, "O": 0.8881}, 75.0, 1.0,
    sternheimer=(3.5017, 0.2400, 2.8004, 0.09116, 3.4773),
)
LUNG = Material(
    "lung",
    {"H": 0.103, "C": 0.105, "N": 0.031, "O": 0.749,
     "Na": 0.002, "P": 0.002, "S": 0.003, "Cl": 0.003, "K": 0.002},
    75.2, 0.26,
)
SOFT = Material(
    "soft_tissue",
    {"H": 0.102, "C": 0.143, "N": 0.034, "O": 0.708,
     "Na": 0.002, "P": 0.003, "S": 0.003, "Cl": 0.002, "K": 0.003},
    74.7, 1.04,
)
BONE = Material(
    "bone",
    {"H": 0.064, "C": 0.278, "N": 0.027, "O": 0.410,
     "Mg": 0.002, "P": 0.070, "S": 0.002, "Ca": 0.147},
    91.9, 1.85,
)
AIR = Material(
    "air", {"C": 0.0001, "N": 0.7553, "O": 0.2318, "Ar": 0.0128}, 85.7, 0.0012, gas=True,
)

BY_NAME = {m.name: m for m in (WATER, LUNG, SOFT, BONE, AIR)}
