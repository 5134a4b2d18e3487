"""Dose-comparison metrics of the paper's evaluation (Sec. II.D), host-side numpy.

Not part of the hot path: these consume finished dose grids.
  gamma_index           Eq. 14-15 (Low & Dempsey), criteria 2 % / 2 mm (L231)
  relative_uncertainty  Eq. 12 (the per-voxel uncertainty comes from Eq. 13 or from a batch estimate of it)
  efficiency            Eq. 11
  batch_mean_sigma      mean and standard error over independent batches
  voxel_agreement       fraction of significant voxels within k combined standard errors
"""
from __future__ import annotations

import numpy as np


def batch_mean_sigma(batches: np.ndarray):
    """batches: [B, ...] independent estimates -> (mean, standard error of the mean)."""
    b = np.asarray(batches, dtype=np.float64)
    mean = b.mean(axis=0)
    sigma = b.std(axis=0, ddof=1) / np.sqrt(b.shape[0])
    return mean, sigma


def relative_uncertainty(dose: np.ndarray, sigma: np.ndarray, frac: float = 0.2) -> float:
    """Eq. 12: mean relative uncertainty over voxels with D > frac * D_max."""
    sel = dose > frac * dose.max()
    return float(np.mean(sigma[sel] / dose[sel]))


def efficiency(s: float, seconds: float) -> float:
    """Eq. 11: epsilon = 1 / (s^2 T)."""
    return 1.0 / (s * s * seconds)


def voxel_agreement(a, sa, b, sb, frac: float = 0.1, k: float = 3.0) -> float:
    """Fraction of voxels with a > frac*max(a) whose difference is within k*sqrt(sa^2+sb^2)."""
    sel = a > frac * a.max()
    tol = k * np.sqrt(sa[sel] ** 2 + sb[sel] ** 2)
    return float(np.mean(np.abs(a[sel] - b[sel]) <= tol))


def gamma_index(ref: np.ndarray, test: np.ndarray, voxel_cm: float, dd_frac: float = 0.02, dta_cm: float = 0.2,
                frac: float = 0.1, search_cm: float = 0.6, sub: int = 10):
    """Gamma index of ``test`` against ``ref`` (Eq. 14-15) on voxels with ref > frac * max(ref).

    Delta D = dd_frac * max(ref) (the paper normalises to D_max, L200).  The search first tries
    x' = x (pure dose difference); voxels that fail are searched on a grid of step voxel/sub inside
    a cube of half-width ``search_cm`` with trilinear interpolation of ``test``.
    Returns (gamma over the selected voxels, boolean selection mask).
    """
    from scipy.ndimage import map_coordinates

    ref = np.asarray(ref, np.float64)
    test = np.asarray(test, np.float64)
    dD = dd_frac * ref.max()
    sel = ref > frac * ref.max()
    idx = np.argwhere(sel)
    g = np.abs(test[sel] - ref[sel]) / dD
    bad = np.nonzero(g > 1.0)[0]
    if bad.size:
        n = int(np.ceil(search_cm / voxel_cm * sub))
        off = np.arange(-n, n + 1) / sub                      # in voxels
        oz, oy, ox = np.meshgrid(off, off, off, indexing="ij")
        dist2 = (oz**2 + oy**2 + ox**2).ravel() * voxel_cm**2 / dta_cm**2
        keep = dist2 <= (search_cm / dta_cm) ** 2
        oz, oy, ox, dist2 = oz.ravel()[keep], oy.ravel()[keep], ox.ravel()[keep], dist2[keep]
        for j in bad:
            z, y, x = idx[j]
            vals = map_coordinates(test, [z + oz, y + oy, x + ox], order=1, mode="nearest")
            gam2 = dist2 + ((vals - ref[z, y, x]) / dD) ** 2
            g[j] = min(g[j], float(np.sqrt(gam2.min())))
    return g, sel


def gamma_pass_rate(ref, test, voxel_cm, **kw) -> float:
    g, _ = gamma_index(ref, test, voxel_cm, **kw)
    return float(np.mean(g <= 1.0))
