"""Gamma index (Low et al. 1998) between two dose grids on the same voxel lattice: global dose criterion
(fraction of the reference maximum), distance-to-agreement in cm, the evaluated grid interpolated trilinearly
on a sub-voxel search lattice.  Test helper; plain numpy."""
import numpy as np
from scipy import ndimage


def gamma_pass_rate(ref, ev, voxel_cm, dose_frac=0.01, dta_cm=0.1, threshold=0.10, step_cm=0.025, max_points=0, seed=0):
    """ref, ev: 3-D arrays (z, y, x).  Returns (pass rate over voxels with ref >= threshold * max, gamma array).
    max_points > 0: evaluate a seeded random sample of that many of those voxels (large grids)."""
    ref = np.asarray(ref, np.float64); ev = np.asarray(ev, np.float64)
    dmax = ref.max()
    idx = np.argwhere(ref >= threshold * dmax)
    if max_points and len(idx) > max_points:
        idx = idx[np.sort(np.random.default_rng(seed).choice(len(idx), max_points, replace=False))]
    dd = dose_frac * dmax
    n = int(np.floor(dta_cm * 1.0001 / step_cm))
    offs = np.arange(-n, n + 1) * step_cm
    best = np.full(len(idx), np.inf)
    base = idx.T.astype(np.float64)
    for oz in offs:
        for oy in offs:
            for ox in offs:
                r2 = oz * oz + oy * oy + ox * ox
                if r2 > dta_cm * dta_cm * 1.0001:
                    continue
                coords = base + np.array([[oz / voxel_cm[2]], [oy / voxel_cm[1]], [ox / voxel_cm[0]]])
                v = ndimage.map_coordinates(ev, coords, order=1, mode="nearest")
                g2 = ((v - ref[tuple(idx.T)]) / dd) ** 2 + (r2 / (dta_cm * dta_cm) if dta_cm > 0 else 0.0)
                best = np.minimum(best, g2)
    gam = np.sqrt(best)
    return float((gam <= 1.0).mean()), gam
