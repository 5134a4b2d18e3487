"""Seeded synthetic phantoms for the five BASELINE.json configs (input data only).

They stand in for the paper's slab phantoms and for the
CT-based phantoms it lists as future work (L389); none of the paper's own
geometry files exist.  Voxel (ix,iy,iz) has linear index ix + nx*(iy + ny*iz);
the beam enters the z=0 face travelling along +z.

Each generator returns (density float32[nz,ny,nx], material uint8[nz,ny,nx]).
"""
from __future__ import annotations

import numpy as np


def homogeneous(nx: int, ny: int, nz: int, density: float = 1.0, material: int = 0):
    rho = np.full((nz, ny, nx), density, dtype=np.float32)
    mat = np.full((nz, ny, nx), material, dtype=np.uint8)
    return rho, mat


def z_slabs(nx: int, ny: int, nz: int, slabs):
    """``slabs`` = [(n_voxels_thick or None for 'rest', density, material_id), ...] stacked along +z."""
    rho = np.empty((nz, ny, nx), dtype=np.float32)
    mat = np.empty((nz, ny, nx), dtype=np.uint8)
    z0 = 0
    for thick, d, m in slabs:
        z1 = nz if thick is None else min(nz, z0 + int(thick))
        rho[z0:z1] = d
        mat[z0:z1] = m
        z0 = z1
    if z0 != nz:
        raise ValueError("slabs do not fill the phantom")
    return rho, mat


def box_in_background(nx: int, ny: int, nz: int, voxel_cm: float, background, box, z0_cm: float, length_cm: float,
                      width_cm: float):
    """A box of (density, material) ``box`` inside a phantom of ``background``, centred on the beam axis
    (the phantom's x-y centre), starting at depth ``z0_cm`` (the paper's lung box).
    A voxel belongs to the box when its centre lies inside it."""
    rho, mat = homogeneous(nx, ny, nz, *background)
    cx, cy = 0.5 * nx * voxel_cm, 0.5 * ny * voxel_cm
    x = (np.arange(nx) + 0.5) * voxel_cm
    y = (np.arange(ny) + 0.5) * voxel_cm
    z = (np.arange(nz) + 0.5) * voxel_cm
    inx = np.abs(x - cx) < 0.5 * width_cm
    iny = np.abs(y - cy) < 0.5 * width_cm
    inz = (z > z0_cm) & (z < z0_cm + length_cm)
    sel = inz[:, None, None] & iny[None, :, None] & inx[None, None, :]
    rho[sel] = box[0]
    mat[sel] = box[1]
    return rho, mat


def ct_like(nx: int, ny: int, nz: int, voxel_cm: float, seed: int = 5, sigma_cm: float = 2.0,
            fractions=(0.10, 0.20, 0.55, 0.15), densities=(0.0012, 0.26, 1.04, 1.85),
            noise: float = 0.03):
    """CT-like phantom of config 5.

    A unit-variance white Gaussian field from ``numpy.random.default_rng(seed)``
    is smoothed with a periodic Gaussian filter (sigma = ``sigma_cm``) applied in
    Fourier space, then thresholded by quantile into air / lung / soft tissue /
    bone (material ids 0..3, lowest field values = air).  Every voxel's density
    is its class density times (1 + u), u ~ Uniform(-noise, +noise) from the
    same generator.
    """
    rng = np.random.default_rng(seed)
    g = rng.standard_normal((nz, ny, nx))
    kz = np.fft.fftfreq(nz, d=voxel_cm)[:, None, None]
    ky = np.fft.fftfreq(ny, d=voxel_cm)[None, :, None]
    kx = np.fft.rfftfreq(nx, d=voxel_cm)[None, None, :]
    filt = np.exp(-2.0 * (np.pi * sigma_cm) ** 2 * (kx**2 + ky**2 + kz**2))
    g = np.fft.irfftn(np.fft.rfftn(g, axes=(0, 1, 2)) * filt, s=g.shape, axes=(0, 1, 2))
    edges = np.quantile(g, np.cumsum(fractions)[:-1])
    mat = np.digitize(g, edges).astype(np.uint8)
    u = rng.uniform(-noise, noise, size=g.shape)
    rho = (np.asarray(densities)[mat] * (1.0 + u)).astype(np.float32)
    return rho, mat
