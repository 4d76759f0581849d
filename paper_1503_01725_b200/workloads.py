"""Seeded synthetic inputs for the PSL source + MC dose path (configs C0..C4 of BASELINE.json).

This module only GENERATES INPUTS (PSR weight tables, jaws, phantoms, beam set-ups); it holds none
of the method's arithmetic and imports neither the CUDA binding nor the oracle.  Both are fed from
here.  The recipe is stated in DESIGN.md §"Inputs"; the TrueBeam-fitted model, patient CTs and
plans the paper measures on are not available, these stand in for them.

numpy only, double precision.
"""
from __future__ import annotations

import math

import numpy as np

R_MAX = 16.0      # cm, radius of the phase-space plane covered by rings
E_MAX = 6.0       # MeV
Z_PHSP = 70.0     # cm
SAD = 100.0       # cm
Z_JY, Z_JX = 76.0, 82.0   # thin jaws, downstream of the phase-space plane
SUBSOURCE_WEIGHT = (0.917, 0.08, 0.003)          # primary, extra-focal photons, electrons
SIGMA_SRC = (0.1, 1.5, 2.0)                      # cm
Z_SRC = (0.0, 12.0, 12.0)                        # cm
PARTICLE_TYPE = (0, 0, 1)                        # photon, photon, electron
WATER, LUNG, BONE = 0, 1, 2


# ---------------------------------------------------------------- PSR model (closed-form integrals)
def _int_E_exp(E, a):
    """Antiderivative of E*exp(-E/a)*(1-E/6)."""
    ex = np.exp(-E / a)
    i1 = -a * ex * (E + a)                              # ∫ E e^{-E/a}
    i2 = -a * ex * (E * E + 2 * a * E + 2 * a * a)      # ∫ E^2 e^{-E/a}
    return i1 - i2 / E_MAX


def _int_exp(E, b):
    """Antiderivative of exp(-E/b)*(1-E/6)."""
    ex = np.exp(-E / b)
    return -b * ex - (-b * ex * (E + b)) / E_MAX


def spectrum_bins(stype: int, n_ebin: int) -> np.ndarray:
    """Normalised bin integrals of the 'Schiff-like' spectra on 0..6 MeV."""
    edges = np.linspace(0.0, E_MAX, n_ebin + 1)
    if stype == 0:
        F = _int_E_exp(edges, 0.9)
    elif stype == 1:
        F = _int_E_exp(edges, 0.5)
    else:
        F = _int_exp(edges, 1.5)
    w = np.diff(F)
    return w / w.sum()


def _int_fluence(r):
    """∫_0^r f(r') r' dr' with f = 1+0.04 r^2 (r<=12), f(12)*(16-r)/4 (12<r<=16)."""
    r = np.asarray(r, dtype=np.float64)
    inner = lambda x: x * x / 2 + 0.01 * x ** 4
    f12 = 1 + 0.04 * 144.0
    outer = lambda x: (f12 / 4) * (8 * x * x - x ** 3 / 3)
    return np.where(r <= 12.0, inner(np.minimum(r, 12.0)), inner(12.0) + outer(r) - outer(12.0))


def fluence_rings(n_ring: int) -> np.ndarray:
    edges = np.linspace(0.0, R_MAX, n_ring + 1)
    w = np.diff(_int_fluence(edges))
    return w / w.sum()


def psr_model(n_ebin: int, n_ring: int) -> dict:
    W = np.empty((3, n_ebin, n_ring), dtype=np.float64)
    F = fluence_rings(n_ring)
    for s in range(3):
        W[s] = SUBSOURCE_WEIGHT[s] * np.outer(spectrum_bins(s, n_ebin), F)
    return dict(n_ebin=n_ebin, n_ring=n_ring, e_min=0.0, e_bin_width=E_MAX / n_ebin,
                ring_width=R_MAX / n_ring, z_phsp=Z_PHSP, W=np.ascontiguousarray(W),
                sigma_src=SIGMA_SRC, z_src=Z_SRC, particle_type=PARTICLE_TYPE)


def direction_model(stype: int, n_ebin: int, n_ring: int) -> dict:
    """Synthetic parameters of the paper's direction models: Eq. 6, K = 3 Gaussians in
    (alpha, beta) per (energy bin, ring) for the scattered photons (stype 1); Eq. 7, one zero-mean Gaussian for the
    electrons (stype 2).  The fitted TrueBeam tables are not available; these follow the geometry of three extended
    virtual sources at z = 12, 25, 45 cm seen from the ring centre, narrowing with energy.  Arrays [n_ebin][n_ring][K]."""
    e = (np.arange(n_ebin) + 0.5) / n_ebin                                  # bin centre / E_max
    r = (np.arange(n_ring) + 0.5) * (R_MAX / n_ring)
    if stype == 1:
        zk = np.array([12.0, 25.0, 45.0]); size = np.array([1.5, 2.5, 4.0]); wk = np.array([0.55, 0.30, 0.15])
        c = np.broadcast_to(wk, (n_ebin, n_ring, 3)) * (1.0 + 0.2 * e[:, None, None] * np.array([1.0, 0.0, -1.0]))
        mu = np.broadcast_to(np.arctan(r[:, None] / (Z_PHSP - zk)[None, :]), (n_ebin, n_ring, 3))
        sig = (size / (Z_PHSP - zk))[None, None, :] * (1.0 - 0.3 * e[:, None, None]) * np.ones((1, n_ring, 1))
        return dict(c=np.ascontiguousarray(c), mu=np.ascontiguousarray(mu), sigma_a=np.ascontiguousarray(sig),
                    sigma_b=np.ascontiguousarray(0.8 * sig))
    if stype == 2:
        sig = 0.06 * (1.0 - 0.4 * e[:, None, None]) * (1.0 + 0.02 * r[None, :, None])
        one = np.ones((n_ebin, n_ring, 1))
        return dict(c=one, mu=0.0 * one, sigma_a=np.ascontiguousarray(sig), sigma_b=np.ascontiguousarray(sig))
    raise ValueError("the primary sub-source keeps the focal model (Eq. 4-5)")


def jaws(field_x: float, field_y: float | None = None) -> dict:
    fy = field_x if field_y is None else field_y
    return dict(x1=-field_x / 2, x2=field_x / 2, y1=-fy / 2, y2=fy / 2, z_jx=Z_JX, z_jy=Z_JY, sad=SAD)


# ---------------------------------------------------------------- beams
def beam_along_z(ssd: float) -> dict:
    """R = I; the beam travels along +z and enters the k = 0 face at z = 0."""
    return dict(iso=(0.0, 0.0, SAD - ssd), R=np.eye(3).reshape(-1).tolist(), sad=SAD)


def beam_gantry(gantry_deg: float) -> dict:
    g = math.radians(gantry_deg)
    bz = (-math.sin(g), -math.cos(g), 0.0)
    bx = (math.cos(g), -math.sin(g), 0.0)
    by = (0.0, 0.0, 1.0)
    R = np.array([bx, by, bz], dtype=np.float64).T      # columns b_x, b_y, b_z
    return dict(iso=(0.0, 0.0, 0.0), R=R.reshape(-1).tolist(), sad=SAD)


# ---------------------------------------------------------------- phantoms
def _phantom(n, d, o, density, material) -> dict:
    return dict(nx=n[0], ny=n[1], nz=n[2], dx=d[0], dy=d[1], dz=d[2], ox=o[0], oy=o[1], oz=o[2],
                density=np.ascontiguousarray(density, dtype=np.float32).reshape(-1),
                material=np.ascontiguousarray(material, dtype=np.uint8).reshape(-1))


def water_cube(n: int, d: float) -> dict:
    shape = (n, n, n)   # (k, j, i) — x fastest
    return _phantom((n, n, n), (d, d, d), (-n * d / 2, -n * d / 2, 0.0),
                    np.ones(shape, np.float32), np.zeros(shape, np.uint8))


def slab_phantom(n: int = 128, d: float = 0.25) -> dict:
    """C2: water 0-3 cm, bone (1.85) 3-5, lung (0.26) 5-12, water beyond, layered along z."""
    zc = (np.arange(n) + 0.5) * d
    rho = np.ones(n, np.float32)
    mat = np.zeros(n, np.uint8)
    bone = (zc >= 3.0) & (zc < 5.0)
    lung = (zc >= 5.0) & (zc < 12.0)
    rho[bone], mat[bone] = 1.85, BONE
    rho[lung], mat[lung] = 0.26, LUNG
    density = np.broadcast_to(rho[:, None, None], (n, n, n))
    material = np.broadcast_to(mat[:, None, None], (n, n, n))
    return _phantom((n, n, n), (d, d, d), (-n * d / 2, -n * d / 2, 0.0), density, material)


def patient_phantom(nx: int = 256, ny: int = 256, nz: int = 120, seed: int = 1003) -> dict:
    """C3: elliptic-cylinder body with two ellipsoidal lungs and a cylindrical spine."""
    d = (0.2, 0.2, 0.25)
    o = (-nx * d[0] / 2, -ny * d[1] / 2, -nz * d[2] / 2)
    x = o[0] + (np.arange(nx) + 0.5) * d[0]
    y = o[1] + (np.arange(ny) + 0.5) * d[1]
    z = o[2] + (np.arange(nz) + 0.5) * d[2]
    Z, Y, X = np.meshgrid(z, y, x, indexing="ij")
    rho = np.full((nz, ny, nx), 0.0012, np.float64)
    body = (X / 15.0) ** 2 + (Y / 10.0) ** 2 <= 1.0
    rho[body] = 1.02
    for cx in (-7.5, 7.5):
        lung = ((X - cx) / 5.0) ** 2 + ((Y - 1.0) / 6.0) ** 2 + (Z / 11.0) ** 2 <= 1.0
        rho[lung & body] = 0.25
    spine = (X ** 2 + (Y + 6.0) ** 2 <= 1.5 ** 2) & body
    rho[spine] = 1.6
    rng = np.random.Generator(np.random.PCG64(seed))
    noise = rng.normal(0.0, 0.01, size=rho.shape)
    rho = np.where(body, np.maximum(rho + noise, 0.001), rho)
    mat = np.where(rho < 0.6, LUNG, np.where(rho <= 1.3, WATER, BONE)).astype(np.uint8)
    return _phantom((nx, ny, nz), d, o, rho, mat)


# ---------------------------------------------------------------- the five configs
GANTRY_C3 = (0, 51, 103, 154, 206, 257, 309)

CONFIGS = {
    "C0": dict(n_ebin=8, n_ring=16, n_sectors=8, field=4.0, ssd=90.0, n_histories=100_000, seed=1,
               phantom=("water", 32, 0.5)),
    "C1": dict(n_ebin=24, n_ring=32, n_sectors=16, field=10.0, ssd=100.0, n_histories=10_000_000, seed=2,
               phantom=("water", 64, 0.25)),
    "C2": dict(n_ebin=24, n_ring=32, n_sectors=16, field=5.0, ssd=100.0, n_histories=100_000_000, seed=3,
               phantom=("slab", 128, 0.25)),
    "C3": dict(n_ebin=24, n_ring=32, n_sectors=16, field=8.0, ssd=None, n_histories=100_000_000, seed=40,
               phantom=("patient",), gantry=GANTRY_C3),
    "C4": dict(n_ebin=48, n_ring=64, n_sectors=32, field=40.0, ssd=100.0, n_histories=1_000_000_000, seed=5,
               phantom=("water", 256, 0.2)),
}


def make_phantom(name: str) -> dict:
    spec = CONFIGS[name]["phantom"]
    if spec[0] == "water":
        return water_cube(spec[1], spec[2])
    if spec[0] == "slab":
        return slab_phantom(spec[1], spec[2])
    return patient_phantom()


def make_config(name: str, with_phantom: bool = True) -> dict:
    """Everything a run of config `name` needs: psr, jaws, n_sectors, beams (list), phantom,
    n_histories (per beam), seed (of beam 0; beam b uses seed + b)."""
    c = CONFIGS[name]
    beams = [beam_gantry(g) for g in c["gantry"]] if "gantry" in c else [beam_along_z(c["ssd"])]
    out = dict(name=name, psr=psr_model(c["n_ebin"], c["n_ring"]), jaws=jaws(c["field"]),
               n_sectors=c["n_sectors"], beams=beams, n_histories=c["n_histories"], seed=c["seed"])
    if with_phantom:
        out["phantom"] = make_phantom(name)
    return out
