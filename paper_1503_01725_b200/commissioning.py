"""Automatic source commissioning (§2.2) — host-side utilities around the GPU tally.

The hot part (the per-PSR dose matrix A) is computed by mc_dose with the commissioning tally (mc_opts_t.com_*:
every history carries the index of the PSR it was sampled from, its descendants inherit it, and deposits in voxels
the 3-D index array marks go to A[column = PSR unit, row = measurement point]).  This module holds what the paper
does on the host: which voxels are measurement points (depth dose on the central axis, in-line and cross-line profiles
at a few depths, §2.2.1), the column numbering (one per photon PSR, one per electron energy bin, §2.2.3) and the
solver of  min_{x >= 0} ||A x - b||^2  (Eq. 8) by gradient projection with Armijo's rule (§2.2.4).
"""
from __future__ import annotations

import numpy as np


def n_columns(n_ebin: int, n_ring: int) -> int:
    """Photon PSRs of the two photon sub-sources + one effective unit per electron energy bin."""
    return 2 * n_ebin * n_ring + n_ebin


def measurement_index(nx: int, ny: int, nz: int, dz: float, depths_cm=(1.5, 10.0, 20.0)) -> tuple[np.ndarray, int]:
    """The 3-D index array of PAPER.md:134: 0 = voxel not needed, otherwise 1 + row.  Rows: the central-axis depth dose
    (nz points), then for each depth the cross-line (x) and the in-line (y) profile through the axis.  The beam
    travels along +z and enters at k = 0; the axis runs through voxel (nx // 2, ny // 2).  Returns (index[nz, ny, nx], rows)."""
    idx = np.zeros((nz, ny, nx), np.int32)
    row = 0
    ic, jc = nx // 2, ny // 2
    for k in range(nz):
        row += 1
        idx[k, jc, ic] = row
    for d in depths_cm:
        k = int(d / dz)
        if not 0 <= k < nz:
            continue
        for i in range(nx):
            if idx[k, jc, i] == 0:
                row += 1
                idx[k, jc, i] = row
        for j in range(ny):
            if idx[k, j, ic] == 0:
                row += 1
                idx[k, j, ic] = row
    return idx, row


def solve_gradient_projection(A: np.ndarray, b: np.ndarray, x0: np.ndarray | None = None, delta: float = 1e-10,
                              max_iter: int = 20000, sigma: float = 1e-4, beta: float = 0.5):
    """Eq. 8: min_{x >= 0} F(x) = ||A x - b||_2^2 by the gradient projection method, x^{k+1} = P(x^k - s_k grad F(x^k)),
    P(y) = max(0, y), with Armijo's rule along the projection arc for s_k; stops when the relative change of F between
    two successive iterations is below `delta`.  Returns (x, info)."""
    A = np.asarray(A, np.float64)
    b = np.asarray(b, np.float64)
    m, n = A.shape
    x = np.ones(n) if x0 is None else np.maximum(0.0, np.asarray(x0, np.float64)).copy()   # correction factors start at 1
    r = A @ x - b
    F = float(r @ r)
    # first trial step: 1 / L with L = 2 ||A||_2^2 (power iteration); afterwards the last accepted step, once enlarged
    v = np.ones(n) / np.sqrt(n)
    for _ in range(30):
        w = A.T @ (A @ v)
        nw = np.linalg.norm(w)
        if nw == 0:
            break
        v = w / nw
    L = 2.0 * float(v @ (A.T @ (A @ v))) if n else 1.0
    s = 1.0 / L if L > 0 else 1.0
    it, evals = 0, 0
    history = [F]
    for it in range(1, max_iter + 1):
        g = 2.0 * (A.T @ r)
        s = s / beta                                       # try a longer step than the one accepted last time
        while True:
            xn = np.maximum(0.0, x - s * g)                # the projection P
            rn = A @ xn - b
            Fn = float(rn @ rn)
            evals += 1
            if Fn <= F - sigma * float(g @ (x - xn)) or s < 1e-300:     # Armijo's rule on the projection arc
                break
            s *= beta
        dF = F - Fn
        x, r, F = xn, rn, Fn
        history.append(F)
        if dF <= delta * max(F, 1e-300) or F == 0.0:
            break
    g = 2.0 * (A.T @ r)
    kkt = float(np.max(np.abs(np.where(x > 0, g, np.minimum(g, 0.0))))) if n else 0.0   # projected-gradient optimality
    return x, dict(iterations=it, evaluations=evals, objective=F, kkt=kkt, history=history)
