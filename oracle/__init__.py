"""ctypes front end of the CPU oracle (oracle/pslmc_oracle.cpp).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference leg may import this.  It imports nothing from
paper_1503_01725_b200 and shares no code with the CUDA path.

Inputs are the plain dicts produced by paper_1503_01725_b200.workloads (the caller passes them).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "pslmc_oracle.cpp")
_LIB = os.path.join(_HERE, "liboracle.so")


def build(force: bool = False) -> str:
    """g++ -O2, no fast-math.  Rebuilds when the source is newer than the library."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".tmp%d" % os.getpid()
        subprocess.check_call(["g++", "-O2", "-std=c++17", "-shared", "-fPIC", "-o", tmp, _SRC])
        os.replace(tmp, _LIB)
    return _LIB


class _Psr(C.Structure):
    _fields_ = [("n_ebin", C.c_int32), ("n_ring", C.c_int32), ("e_min", C.c_double), ("e_bin_width", C.c_double),
                ("ring_width", C.c_double), ("z_phsp", C.c_double), ("W", C.POINTER(C.c_double)),
                ("sigma_src", C.c_double * 3), ("z_src", C.c_double * 3), ("particle_type", C.c_int32 * 3)]


class _Jaws(C.Structure):
    _fields_ = [(k, C.c_double) for k in ("x1", "x2", "y1", "y2", "z_jx", "z_jy", "sad")]


class _Phantom(C.Structure):
    _fields_ = [("nx", C.c_int32), ("ny", C.c_int32), ("nz", C.c_int32)] + \
               [(k, C.c_double) for k in ("dx", "dy", "dz", "ox", "oy", "oz")] + \
               [("density", C.c_void_p), ("material", C.c_void_p)]


class _Beam(C.Structure):
    _fields_ = [("iso", C.c_double * 3), ("R", C.c_double * 9), ("sad", C.c_double)]


class _Result(C.Structure):
    _fields_ = [("ledger_hi", C.c_int64 * 4), ("ledger_lo", C.c_uint64 * 4), ("n_hist", C.c_uint64 * 3)] + \
               [(k, C.c_uint64) for k in (
                   "n_jaw_rejected", "n_missed", "n_flights", "n_virtual", "n_compton", "n_photo", "n_pair",
                   "n_photon_cutoff", "n_photon_escape", "n_uncollided_escape", "n_sec_electrons", "n_sec_photons",
                   "n_electron_tracks", "n_electron_steps", "n_electron_escape", "n_deposits", "n_kahn_trials", "n_deflections")]


LEDGERS = ("incident", "deposited", "escaped", "jaw")
FLAG_ELECTRONS_LOCAL, FLAG_TRACE_BIRTH, FLAG_FP_VOXELS = 1, 2, 4      # orc_dose / orc_transport / orc_trace flags
_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        L.orc_psl_build.restype = C.c_void_p
        L.orc_psl_build.argtypes = [C.POINTER(_Psr), C.POINTER(_Jaws), C.c_int32]
        L.orc_psl_build_grid.restype = C.c_void_p
        L.orc_psl_build_grid.argtypes = [C.POINTER(_Psr), C.POINTER(_Jaws), C.c_double]
        L.orc_psl_grid_n.argtypes = [C.c_void_p]
        L.orc_psl_grid_x0.restype = C.c_double
        L.orc_psl_grid_x0.argtypes = [C.c_void_p]
        L.orc_psl_set_direction.argtypes = [C.c_void_p, C.c_int32, C.c_int32] + [C.c_void_p] * 4
        L.orc_psl_free.argtypes = [C.c_void_p]
        L.orc_psl_n_groups.argtypes = [C.c_void_p]
        L.orc_psl_group_size.restype = C.c_int64
        L.orc_psl_group_size.argtypes = [C.c_void_p, C.c_int32]
        L.orc_psl_group_weight.restype = C.c_double
        L.orc_psl_group_weight.argtypes = [C.c_void_p, C.c_int32]
        L.orc_psl_group_get.argtypes = [C.c_void_p, C.c_int32] + [C.c_void_p] * 4
        L.orc_psl_rect.argtypes = [C.c_void_p, C.c_void_p]
        L.orc_allocate.argtypes = [C.c_void_p, C.c_uint64, C.c_void_p]
        L.orc_sample.argtypes = [C.c_void_p, C.POINTER(_Beam), C.c_uint64, C.c_uint64, C.c_uint64, C.c_uint64, C.c_void_p]
        L.orc_dose.argtypes = [C.c_void_p, C.POINTER(_Phantom), C.POINTER(_Beam), C.c_uint64, C.c_uint64, C.c_uint64,
                               C.c_uint64, C.c_int32, C.c_void_p, C.POINTER(_Result), C.c_void_p]
        L.orc_dose_list.argtypes = [C.c_void_p, C.POINTER(_Phantom), C.POINTER(_Beam), C.c_uint64, C.c_uint64, C.c_void_p,
                                    C.c_uint64, C.c_int32, C.c_void_p, C.POINTER(_Result), C.c_void_p]
        L.orc_dose_com.argtypes = [C.c_void_p, C.POINTER(_Phantom), C.POINTER(_Beam), C.c_uint64, C.c_uint64, C.c_uint64,
                                   C.c_uint64, C.c_void_p, C.POINTER(_Result), C.c_void_p, C.c_void_p, C.c_int64]
        L.orc_com_column.restype = C.c_uint32
        L.orc_com_column.argtypes = [C.c_int32] * 6
        L.orc_transport.argtypes = [C.POINTER(_Phantom), C.c_int32, C.c_void_p, C.c_uint64, C.c_uint64, C.c_uint64,
                                    C.c_int32, C.c_double, C.c_void_p, C.POINTER(_Result), C.c_void_p]
        L.orc_trace.argtypes = [C.POINTER(_Phantom), C.c_int32, C.c_void_p, C.c_uint64, C.c_uint64, C.c_int32,
                                C.c_double, C.c_void_p, C.c_int32]
        L.orc_philox.argtypes = [C.c_uint64, C.c_uint64, C.c_uint32, C.c_uint32, C.c_void_p]
        L.orc_child_track.restype = C.c_uint32
        L.orc_child_track.argtypes = [C.c_uint32] * 3
        L.orc_sigma_kn.restype = C.c_double
        L.orc_sigma_kn.argtypes = [C.c_double]
        L.orc_mu_over_rho.argtypes = [C.c_int32, C.c_double, C.c_void_p]
        L.orc_stopping.restype = C.c_double
        L.orc_stopping.argtypes = [C.c_int32, C.c_double]
        L.orc_kahn.argtypes = [C.c_double, C.c_uint64, C.c_uint64, C.c_uint64, C.c_void_p, C.c_void_p]
        L.orc_rotate.argtypes = [C.c_void_p, C.c_double, C.c_double, C.c_double]
        L.orc_finalise.argtypes = [C.POINTER(_Phantom), C.c_void_p, C.c_uint64, C.c_void_p]
        _lib = L
    return _lib


def _ptr(a: np.ndarray):
    return a.ctypes.data_as(C.c_void_p)


def _beam(b: dict) -> _Beam:
    return _Beam((C.c_double * 3)(*b["iso"]), (C.c_double * 9)(*b["R"]), b["sad"])


class Phantom:
    """Keeps the numpy arrays alive next to the C struct."""

    def __init__(self, ph: dict):
        self.density = np.ascontiguousarray(ph["density"], np.float32)
        self.material = np.ascontiguousarray(ph["material"], np.uint8)
        self.n = (ph["nx"], ph["ny"], ph["nz"])
        self.nvox = ph["nx"] * ph["ny"] * ph["nz"]
        assert self.density.size == self.nvox and self.material.size == self.nvox
        self.c = _Phantom(ph["nx"], ph["ny"], ph["nz"], ph["dx"], ph["dy"], ph["dz"], ph["ox"], ph["oy"], ph["oz"],
                          self.density.ctypes.data, self.material.ctypes.data)


def _result(r: _Result) -> dict:
    out = {k: int(getattr(r, k)) for k, t in _Result._fields_ if t is C.c_uint64}
    out["n_hist"] = [int(x) for x in r.n_hist]
    out["ledger"] = {name: (int(r.ledger_hi[i]) << 64) + int(r.ledger_lo[i]) for i, name in enumerate(LEDGERS)}
    return out


class Psl:
    def __init__(self, psr: dict, jaws: dict, n_sectors: int, let_size: float = 0.0):
        """n_sectors >= 1: ring-sector lets.  n_sectors == 0 and let_size > 0: the paper's Cartesian (Xbin, Ybin) lets
        (PAPER.md:39-55); group()['ring'] / ['sector'] then hold Xbin / Ybin."""
        self._W = np.ascontiguousarray(psr["W"], np.float64)
        p = _Psr(psr["n_ebin"], psr["n_ring"], psr["e_min"], psr["e_bin_width"], psr["ring_width"], psr["z_phsp"],
                 self._W.ctypes.data_as(C.POINTER(C.c_double)), (C.c_double * 3)(*psr["sigma_src"]),
                 (C.c_double * 3)(*psr["z_src"]), (C.c_int32 * 3)(*psr["particle_type"]))
        j = _Jaws(*(jaws[k] for k in ("x1", "x2", "y1", "y2", "z_jx", "z_jy", "sad")))
        if n_sectors == 0:
            self.h = lib().orc_psl_build_grid(C.byref(p), C.byref(j), float(let_size))
        else:
            self.h = lib().orc_psl_build(C.byref(p), C.byref(j), n_sectors)
        if not self.h:
            raise ValueError("empty field: no active let")
        self.n_ebin, self.n_sectors = psr["n_ebin"], n_sectors
        self.n_groups = lib().orc_psl_n_groups(self.h)
        self.let_size = float(let_size)
        self.grid_n = lib().orc_psl_grid_n(self.h) if n_sectors == 0 else 0
        self.grid_x0 = lib().orc_psl_grid_x0(self.h) if n_sectors == 0 else 0.0

    def __del__(self):
        if getattr(self, "h", None) and _lib is not None:        # (at interpreter shutdown the module globals may be gone)
            _lib.orc_psl_free(self.h)
            self.h = None

    def set_direction_model(self, stype: int, c, mu, sigma_a, sigma_b):
        """Eq. 6 / Eq. 7: arrays [n_ebin][n_ring][K] of component weights, means of alpha, sigmas."""
        arrs = [np.ascontiguousarray(a, np.float64) for a in (c, mu, sigma_a, sigma_b)]
        K = arrs[0].shape[-1]
        assert all(a.shape == arrs[0].shape for a in arrs)
        lib().orc_psl_set_direction(self.h, stype, K, *[_ptr(a) for a in arrs])

    def group(self, g: int) -> dict:
        n = lib().orc_psl_group_size(self.h, g)
        ring, sector = np.empty(n, np.uint16), np.empty(n, np.uint16)
        thresh, alias = np.empty(n, np.uint32), np.empty(n, np.uint32)
        lib().orc_psl_group_get(self.h, g, _ptr(ring), _ptr(sector), _ptr(thresh), _ptr(alias))
        return dict(stype=g // self.n_ebin, ebin=g % self.n_ebin, ring=ring, sector=sector, thresh=thresh,
                    alias=alias, W=lib().orc_psl_group_weight(self.h, g))

    def rect(self) -> np.ndarray:
        out = np.empty((3, 4), np.float64)
        lib().orc_psl_rect(self.h, _ptr(out))
        return out

    def allocate(self, n_histories: int) -> np.ndarray:
        off = np.empty(self.n_groups + 1, np.uint64)
        lib().orc_allocate(self.h, n_histories, _ptr(off))
        return off

    def sample(self, beam: dict, n_histories: int, seed: int, first: int, count: int) -> np.ndarray:
        """(count, 8) float64: x, y, z, u, v, w, E, status."""
        out = np.empty((count, 8), np.float64)
        lib().orc_sample(self.h, C.byref(_beam(beam)), n_histories, seed, first, count, _ptr(out))
        return out

    def dose(self, phantom: Phantom, beam: dict, n_histories: int, seed: int, h_begin: int = 0, h_end: int | None = None,
             flags: int = 0, acc: np.ndarray | None = None, fingerprints: bool = False):
        """Returns (acc int64[nvox], result dict, fingerprints u64 or None)."""
        h_end = n_histories if h_end is None else h_end
        if acc is None:
            acc = np.zeros(phantom.nvox, np.int64)
        fp = np.zeros(h_end - h_begin, np.uint64) if fingerprints else None
        res = _Result()
        lib().orc_dose(self.h, C.byref(phantom.c), C.byref(_beam(beam)), n_histories, seed, h_begin, h_end, flags,
                       _ptr(acc), C.byref(res), _ptr(fp) if fp is not None else None)
        return acc, _result(res), fp


def dose_list(psl: "Psl", phantom: Phantom, beam: dict, n_histories: int, seed: int, ids, flags: int = 0,
              acc: np.ndarray | None = None, fingerprints: bool = False):
    """The tally of a list of history ids of an n_histories allocation.  Returns (acc, result dict, fingerprints or None)."""
    ids = np.ascontiguousarray(ids, np.uint64)
    if acc is None:
        acc = np.zeros(phantom.nvox, np.int64)
    fp = np.zeros(ids.size, np.uint64) if fingerprints else None
    res = _Result()
    lib().orc_dose_list(psl.h, C.byref(phantom.c), C.byref(_beam(beam)), n_histories, seed, _ptr(ids), ids.size, flags,
                        _ptr(acc), C.byref(res), _ptr(fp) if fp is not None else None)
    return acc, _result(res), fp


def dose_com(psl: "Psl", phantom: Phantom, beam: dict, n_histories: int, seed: int, com_index: np.ndarray, n_rows: int,
             n_cols: int, h_begin: int = 0, h_end: int | None = None):
    """Dose with the commissioning tally.  Returns (acc int64[nvox], A int64[n_cols, n_rows], result)."""
    h_end = n_histories if h_end is None else h_end
    acc = np.zeros(phantom.nvox, np.int64)
    A = np.zeros((n_cols, n_rows), np.int64)
    idx = np.ascontiguousarray(com_index, np.int32)
    res = _Result()
    lib().orc_dose_com(psl.h, C.byref(phantom.c), C.byref(_beam(beam)), n_histories, seed, h_begin, h_end, _ptr(acc),
                       C.byref(res), _ptr(idx), _ptr(A), n_rows)
    return acc, A, _result(res)


def com_column(n_ebin: int, n_ring: int, particle_type: int, s: int, e: int, r: int) -> int:
    return int(lib().orc_com_column(n_ebin, n_ring, particle_type, s, e, r))


def transport(phantom: Phantom, ptype: int, particles: np.ndarray, first: int, seed: int, flags: int = 0,
              f_e: float = 0.0, acc: np.ndarray | None = None, fingerprints: bool = False):
    particles = np.ascontiguousarray(particles, np.float64)
    count = particles.shape[0]
    if acc is None:
        acc = np.zeros(phantom.nvox, np.int64)
    fp = np.zeros(count, np.uint64) if fingerprints else None
    res = _Result()
    lib().orc_transport(C.byref(phantom.c), ptype, _ptr(particles), first, count, seed, flags, f_e, _ptr(acc),
                        C.byref(res), _ptr(fp) if fp is not None else None)
    return acc, _result(res), fp


def trace(phantom: Phantom, ptype: int, particle, history: int, seed: int, flags: int = 0, f_e: float = 0.0,
          max_events: int = 4096) -> list[dict]:
    particle = np.ascontiguousarray(particle, np.float64)
    ev = np.zeros((max_events, 10), np.float64)
    n = lib().orc_trace(C.byref(phantom.c), ptype, _ptr(particle), history, seed, flags, f_e, _ptr(ev), max_events)
    return [dict(track=int(e[0]), code=chr(int(e[1])), pos=e[2:5].copy(), dir=e[5:8].copy(), E=e[8], aux=e[9])
            for e in ev[:min(n, max_events)]]


def philox(seed: int, h: int, track: int, block: int) -> np.ndarray:
    out = np.empty(4, np.uint32)
    lib().orc_philox(seed, h, track, block, _ptr(out))
    return out


def child_track(parent: int, n: int, c: int) -> int:
    return int(lib().orc_child_track(parent, n, c))


def sigma_kn(E: float) -> float:
    return lib().orc_sigma_kn(E)


def mu_over_rho(m: int, E: float) -> np.ndarray:
    out = np.empty(3, np.float64)
    lib().orc_mu_over_rho(m, E, _ptr(out))
    return out


def stopping(m: int, T: float) -> float:
    return lib().orc_stopping(m, T)


def kahn(E: float, seed: int, first: int, count: int):
    c, e = np.empty(count, np.float64), np.empty(count, np.float64)
    lib().orc_kahn(E, seed, first, count, _ptr(c), _ptr(e))
    return c, e


def rotate(d, ct: float, st: float, phi: float) -> np.ndarray:
    d = np.array(d, np.float64)
    lib().orc_rotate(_ptr(d), ct, st, phi)
    return d


def finalise(phantom: Phantom, acc: np.ndarray, n_histories: int) -> np.ndarray:
    dose = np.empty(phantom.nvox, np.float64)
    lib().orc_finalise(C.byref(phantom.c), _ptr(acc), n_histories, _ptr(dose))
    return dose
