"""The five BASELINE.json workloads as concrete synthetic inputs (data only).

``make_config(i)`` returns everything a transport implementation needs: the
phantom, the table bundle, the source description, the number of histories and
the seed.  ``scale`` shrinks the history count (parity tests run the oracle on
a bounded sample); the geometry is never changed.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from functools import lru_cache
from typing import Optional

import numpy as np

from . import materials as M
from . import phantoms, spectra
from .tables import TableBundle, build_tables

PHOTON, ELECTRON = 0, 1
PENCIL, RECTANGLE, PHASE_SPACE = 0, 1, 2


@dataclass
class Source:
    particle: int
    shape: int
    cx: float
    cy: float
    wx: float = 0.0
    wy: float = 0.0
    energy: float = 0.0
    spec_edges: Optional[np.ndarray] = None    # float32[n+1]
    spec_weights: Optional[np.ndarray] = None  # float32[n]
    phsp: Optional[np.ndarray] = None          # shape PHASE_SPACE: float32[n, 8] {x, y, z, u, v, w, E, type}


@dataclass
class Workload:
    name: str
    density: np.ndarray        # float32 [nz, ny, nx]
    material: np.ndarray       # uint8   [nz, ny, nx]
    voxel_cm: float
    tables: TableBundle
    source: Source
    n_histories: int
    seed: int
    notes: str = ""

    @property
    def shape_xyz(self):
        nz, ny, nx = self.density.shape
        return nx, ny, nz


@lru_cache(maxsize=None)
def _tables(names: tuple) -> TableBundle:
    return build_tables([M.BY_NAME[n] for n in names])


def make_config(i: int, n_histories: Optional[int] = None) -> Workload:
    if i == 1:
        rho, mat = phantoms.homogeneous(32, 32, 32, 1.0, 0)
        # pencil beam at the centre of voxel (16,16): the geometric centre 8.0 cm is a voxel face
        src = Source(PHOTON, PENCIL, 8.25, 8.25, energy=2.0)
        w = Workload("cfg1_2MeV_photon_pencil_water32", rho, mat, 0.5, _tables(("water",)), src, 100_000, 1)
    elif i == 2:
        rho, mat = phantoms.homogeneous(128, 128, 128, 1.0, 0)
        src = Source(ELECTRON, RECTANGLE, 16.0, 16.0, 10.0, 10.0, energy=15.0)
        w = Workload("cfg2_15MeV_electron_10x10_water128", rho, mat, 0.25, _tables(("water",)), src, 1_000_000, 2)
    elif i == 3:
        rho, mat = phantoms.homogeneous(128, 128, 128, 1.0, 0)
        src = Source(PHOTON, RECTANGLE, 16.0, 16.0, 10.0, 10.0, energy=15.0)
        w = Workload("cfg3_15MeV_photon_10x10_water128", rho, mat, 0.25, _tables(("water",)), src, 4_000_000, 3)
    elif i == 4:
        # water 3 cm / bone 2 cm / lung 7 cm / water rest, 0.25 cm voxels
        rho, mat = phantoms.z_slabs(128, 128, 128, [(12, 1.0, 0), (8, 1.85, 1), (28, 0.26, 2), (None, 1.0, 0)])
        src = Source(PHOTON, RECTANGLE, 16.0, 16.0, 5.0, 5.0, energy=6.0)
        w = Workload("cfg4_6MeV_photon_5x5_slabs128", rho, mat, 0.25, _tables(("water", "bone", "lung")), src,
                     20_000_000, 4)
    elif i == 5:
        rho, mat = phantoms.ct_like(256, 256, 128, 0.2, seed=5)
        edges, weights = spectra.thick_target_spectrum(18.0, 0.1, 512)
        src = Source(PHOTON, RECTANGLE, 25.6, 25.6, 10.0, 10.0, spec_edges=edges, spec_weights=weights)
        w = Workload("cfg5_18MV_photon_10x10_ctlike256", rho, mat, 0.2,
                     _tables(("air", "lung", "soft_tissue", "bone")), src, 100_000_000, 5)
    else:
        raise ValueError("config index must be 1..5")
    if n_histories is not None:
        w.n_histories = int(n_histories)
    return w


def make_paper_geometry(geom: int, particle: int, n_histories: Optional[int] = None) -> Workload:
    """The paper's own benchmark cases (Tab. IV-VI): a 64^3 grid of 0.5 cm voxels,
    a 15 MeV monoenergetic parallel beam, 1e6 histories for electrons and 4e6 for photons.
      geom 1: water;
      geom 2: water with a lung box on the axis (electrons: 4 cm long, 4.5 cm wide, from 3 cm depth;
              photons: 6.5 cm long, 4.5 cm wide, from 5.5 cm);
      geom 3: slabs (electrons: 2 cm soft tissue, 2 cm lung, 2 cm bone, soft tissue; photons: 3 cm soft
              tissue, 2 cm lung, 7 cm bone, soft tissue; the text's order, L262-264).
    The paper does not give the field size: 5 x 5 cm^2 is taken (its Tab. I counts ~120 voxels above 0.2 D_max
    per depth slice).  Materials are this repository's synthetic ones (materials.py)."""
    if geom not in (1, 2, 3) or particle not in (PHOTON, ELECTRON):
        raise ValueError("geom must be 1, 2 or 3 and particle PHOTON or ELECTRON")
    n, h = 64, 0.5
    e = particle == ELECTRON
    if geom == 1:
        rho, mat = phantoms.homogeneous(n, n, n, 1.0, 0)
        names = ("water",)
    elif geom == 2:
        z0, length = (3.0, 4.0) if e else (5.5, 6.5)
        rho, mat = phantoms.box_in_background(n, n, n, h, (1.0, 0), (0.26, 1), z0, length, 4.5)
        names = ("water", "lung")
    else:
        slabs = [(4, 1.04, 0), (4, 0.26, 1), (4, 1.85, 2), (None, 1.04, 0)] if e else \
                [(6, 1.04, 0), (4, 0.26, 1), (14, 1.85, 2), (None, 1.04, 0)]
        rho, mat = phantoms.z_slabs(n, n, n, slabs)
        names = ("soft_tissue", "lung", "bone")
    src = Source(particle, RECTANGLE, 16.0, 16.0, 5.0, 5.0, energy=15.0)
    w = Workload(f"paper_geom{geom}_15MeV_{'electron' if e else 'photon'}_64", rho, mat, h, _tables(names), src,
                 1_000_000 if e else 4_000_000, 10 * geom + particle)
    if n_histories is not None:
        w.n_histories = int(n_histories)
    return w
