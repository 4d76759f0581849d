"""Thin ctypes binding of libpslmc (include/pslmc.h): argument marshalling only — every step of the
path runs in the library's CUDA kernels.  torch is used for device memory and streams.

There is no CPU fallback: if libpslmc.so is missing or fails to load, importing succeeds but every
call raises.  The oracle (oracle/) is test infrastructure and is never imported here.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libpslmc.so")

MC_ORDER_SORTED, MC_ORDER_MIXED = 0, 1
MC_FLAG_ELECTRONS_LOCAL, MC_FLAG_STATS, MC_FLAG_TIMING, MC_FLAG_STATIC_LANES, MC_FLAG_STAGE_SCORING = 1, 2, 4, 8, 16
MC_FLAG_RANGE, MC_FLAG_NO_TILE_SORT, MC_FLAG_TILE_SORT, MC_FLAG_FP_VOXELS = 32, 64, 128, 256
LEDGERS = ("incident", "deposited", "escaped", "jaw")
KERNEL_CLASSES = ("sample", "photon", "electron", "finalise", "aux")
EXPORTS = ("psl_build", "psl_build_grid", "psl_set_direction_model", "mc_plan_allocate", "mc_plan_dose", "psl_free", "psl_export", "psl_allocate",
           "mc_workspace_bytes", "mc_host_workspace_bytes", "mc_dose", "mc_dose_host", "mc_dose_static", "mc_static_workspace_bytes",
           "mc_stats", "mc_last_error", "mc_sample_debug", "mc_transport_debug", "mc_philox_debug", "mc_xs_debug")


class PslmcError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__("libpslmc error %d: %s" % (code, msg))
        self.code = code


class psr_params_t(C.Structure):
    _fields_ = [("n_ebin", C.c_int32), ("n_ring", C.c_int32), ("e_min", C.c_double), ("e_bin_width", C.c_double),
                ("ring_width", C.c_double), ("z_phsp", C.c_double), ("W", C.POINTER(C.c_double)),
                ("sigma_src", C.c_double * 3), ("z_src", C.c_double * 3), ("particle_type", C.c_int32 * 3)]


class jaws_t(C.Structure):
    _fields_ = [(k, C.c_double) for k in ("x1", "x2", "y1", "y2", "z_jx", "z_jy", "sad")]


class phantom_t(C.Structure):
    _fields_ = [("nx", C.c_int32), ("ny", C.c_int32), ("nz", C.c_int32)] + \
               [(k, C.c_double) for k in ("dx", "dy", "dz", "ox", "oy", "oz")] + \
               [("density", C.c_void_p), ("material", C.c_void_p)]


class beam_geom_t(C.Structure):
    _fields_ = [("iso", C.c_double * 3), ("R", C.c_double * 9), ("sad", C.c_double)]


class mc_opts_t(C.Structure):
    _fields_ = [("workspace", C.c_void_p), ("workspace_bytes", C.c_size_t), ("cuda_stream", C.c_void_p),
                ("dose_acc", C.c_void_p), ("order", C.c_int32), ("flags", C.c_int32), ("fingerprints", C.c_void_p),
                ("history_begin", C.c_uint64), ("history_end", C.c_uint64), ("pipelines", C.c_int32), ("reserved", C.c_int32),
                ("com_index", C.c_void_p), ("com_dose", C.c_void_p), ("com_rows", C.c_int32), ("com_cols", C.c_int32),
                ("aux_streams", C.c_void_p * 2), ("shard_index", C.c_int32), ("shard_count", C.c_int32),
                ("debug_eq_cap", C.c_uint32), ("reserved2", C.c_uint32)]


class mc_stats_t(C.Structure):
    _fields_ = [("ledger_hi", C.c_int64 * 4), ("ledger_lo", C.c_uint64 * 4), ("n_hist", C.c_uint64 * 3)] + \
               [(k, C.c_uint64) for k in (
                   "n_jaw_rejected", "n_missed", "n_flights", "n_virtual", "n_compton", "n_photo", "n_pair",
                   "n_photon_cutoff", "n_photon_escape", "n_uncollided_escape", "n_sec_electrons", "n_sec_photons",
                   "n_electron_tracks", "n_electron_steps", "n_electron_escape", "n_deposits", "n_kahn_trials",
                   "n_deflections", "queue_high_water")] + \
               [("launches", C.c_uint64 * 5), ("ms", C.c_float * 5),
                ("ms_total", C.c_float)]


_lib = None


def lib():
    """Loads libpslmc.so (never builds it, never falls back)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError("libpslmc.so not built: run `python -m paper_1503_01725_b200.build` "
                              "(or __graft_entry__.build()); there is no CPU fallback")
        L = C.CDLL(LIB_PATH)
        L.psl_build.argtypes = [C.POINTER(psr_params_t), C.POINTER(jaws_t), C.c_int32, C.POINTER(C.c_void_p)]
        L.psl_build_grid.argtypes = [C.POINTER(psr_params_t), C.POINTER(jaws_t), C.c_double, C.POINTER(C.c_void_p)]
        L.mc_plan_allocate.argtypes = [C.c_void_p, C.c_int32, C.c_uint64, C.c_void_p]
        L.psl_set_direction_model.argtypes = [C.c_void_p, C.c_int32, C.c_int32] + [C.c_void_p] * 4
        L.psl_free.argtypes = [C.c_void_p]
        L.psl_free.restype = None
        L.psl_export.argtypes = [C.c_void_p, C.c_void_p, C.POINTER(C.c_size_t)]
        L.psl_allocate.argtypes = [C.c_void_p, C.c_uint64, C.c_void_p]
        for f in (L.mc_workspace_bytes, L.mc_host_workspace_bytes):
            f.restype = C.c_size_t
            f.argtypes = [C.c_void_p, C.POINTER(phantom_t), C.c_uint64]
        L.mc_plan_dose.argtypes = [C.c_void_p, C.c_void_p, C.c_int32, C.POINTER(phantom_t), C.c_uint64, C.c_uint64, C.c_uint64,
                                   C.c_void_p, C.POINTER(mc_opts_t), C.c_void_p]
        dose_args = [C.c_void_p, C.POINTER(phantom_t), C.POINTER(beam_geom_t), C.c_uint64, C.c_uint64, C.c_uint64,
                     C.c_void_p, C.POINTER(mc_opts_t)]
        L.mc_dose.argtypes = dose_args
        L.mc_dose_host.argtypes = dose_args
        L.mc_dose_static.argtypes = dose_args
        L.mc_static_workspace_bytes.restype = C.c_size_t
        L.mc_static_workspace_bytes.argtypes = []
        L.mc_stats.argtypes = [C.POINTER(mc_stats_t)]
        L.mc_last_error.restype = C.c_char_p
        L.mc_sample_debug.argtypes = [C.c_void_p, C.POINTER(beam_geom_t), C.c_uint64, C.c_uint64, C.c_uint64, C.c_uint64,
                                      C.c_void_p, C.c_void_p]
        L.mc_transport_debug.argtypes = [C.POINTER(phantom_t), C.c_int32, C.c_void_p, C.c_uint64, C.c_uint64, C.c_uint64,
                                         C.POINTER(mc_opts_t)]
        L.mc_philox_debug.argtypes = [C.c_uint64, C.c_uint64, C.c_uint32, C.c_uint32, C.c_void_p]
        L.mc_xs_debug.argtypes = [C.c_void_p, C.c_double, C.c_void_p, C.c_uint64, C.c_void_p]
        _lib = L
    return _lib


def _check(rc: int):
    if rc != 0:
        raise PslmcError(rc, lib().mc_last_error().decode())


def _beam(b: dict) -> beam_geom_t:
    return beam_geom_t((C.c_double * 3)(*b["iso"]), (C.c_double * 9)(*b["R"]), b["sad"])


def _stream_ptr(stream) -> int:
    if stream is None:
        import torch
        stream = torch.cuda.current_stream()
    return int(stream.cuda_stream)


def _phantom_struct(ph: dict, density_ptr: int, material_ptr: int) -> phantom_t:
    return phantom_t(ph["nx"], ph["ny"], ph["nz"], ph["dx"], ph["dy"], ph["dz"], ph["ox"], ph["oy"], ph["oz"],
                     density_ptr, material_ptr)


class DevicePhantom:
    """A phantom resident in HBM (torch tensors own the memory)."""

    def __init__(self, ph: dict, device="cuda:0"):
        import torch
        self.meta = {k: ph[k] for k in ("nx", "ny", "nz", "dx", "dy", "dz", "ox", "oy", "oz")}
        self.nvox = ph["nx"] * ph["ny"] * ph["nz"]
        self.density = torch.as_tensor(np.ascontiguousarray(ph["density"], np.float32)).to(device)
        self.material = torch.as_tensor(np.ascontiguousarray(ph["material"], np.uint8)).to(device)
        assert self.density.numel() == self.nvox and self.material.numel() == self.nvox
        self.c = _phantom_struct(self.meta, self.density.data_ptr(), self.material.data_ptr())
        self.device = self.density.device


def stats() -> dict:
    s = mc_stats_t()
    _check(lib().mc_stats(C.byref(s)))
    out = {k: int(getattr(s, k)) for k, t in mc_stats_t._fields_ if t is C.c_uint64}
    out["n_hist"] = [int(x) for x in s.n_hist]
    out["ledger"] = {n: (int(s.ledger_hi[i]) << 64) + int(s.ledger_lo[i]) for i, n in enumerate(LEDGERS)}
    out["launches"] = {n: int(s.launches[i]) for i, n in enumerate(KERNEL_CLASSES)}
    out["ms"] = {n: float(s.ms[i]) for i, n in enumerate(KERNEL_CLASSES)}
    out["ms_total"] = float(s.ms_total)
    return out


DEFAULT_BATCH = 1 << 24        # histories per k_sample launch: 13.3 GB of workspace (3 pipelines x 264 B), measured best on C1-C4
_aux = {}                                                # device index -> two torch streams for the pipelines (torch owns them)
_ws = {}                                                 # device index -> cached torch workspace (torch owns the memory)


def aux_streams(device=None):
    import torch
    d = torch.cuda.current_device() if device is None else torch.device(device).index
    if d not in _aux:
        _aux[d] = (torch.cuda.Stream(device=d), torch.cuda.Stream(device=d))
    return _aux[d]


def workspace(nbytes: int, device=None):
    """A torch uint8 tensor of at least nbytes on the device, cached and grown on demand (the library never allocates)."""
    import torch
    d = torch.cuda.current_device() if device is None else torch.device(device).index
    t = _ws.get(d)
    if t is None or t.numel() < nbytes:
        _ws[d] = None
        t = _ws[d] = torch.empty(nbytes, dtype=torch.uint8, device="cuda:%d" % d)
    return t


def _opts(stream=None, workspace=None, dose_acc=None, order=0, flags=0, fingerprints=None, history_begin=None,
          history_end=None, pipelines=0, com_index=None, com_dose=None, shard=None, debug_eq_cap=0, aux=None) -> mc_opts_t:
    o = mc_opts_t()
    if workspace is not None:
        o.workspace, o.workspace_bytes = workspace.data_ptr(), workspace.numel() * workspace.element_size()
    o.cuda_stream = _stream_ptr(stream)
    o.dose_acc = dose_acc.data_ptr() if dose_acc is not None else None
    o.order, o.flags = order, flags
    o.fingerprints = fingerprints.data_ptr() if fingerprints is not None else None
    if history_begin is not None or history_end is not None:       # an explicit range is taken literally ([0, 0) is empty)
        o.history_begin, o.history_end = history_begin or 0, history_end or 0
        if history_end is not None:
            o.flags |= MC_FLAG_RANGE
    o.pipelines = pipelines
    if pipelines != 1:
        a = aux if aux is not None else aux_streams()
        o.aux_streams[0], o.aux_streams[1] = int(a[0].cuda_stream), int(a[1].cuda_stream)
    if com_index is not None:                            # commissioning tally: int32[nvox] index, int64[cols, rows] matrix (torch, device)
        o.com_index, o.com_dose = com_index.data_ptr(), com_dose.data_ptr()
        o.com_cols, o.com_rows = com_dose.shape[0], com_dose.shape[1]
    if shard is not None:
        o.shard_index, o.shard_count = shard
    o.debug_eq_cap = debug_eq_cap
    return o


class Psl:
    """psl_build handle: active lets + alias tables, on the host and uploaded to the current device."""

    def __init__(self, psr: dict, jaws: dict, n_sectors: int, let_size: float = 0.0):
        """n_sectors >= 1: ring-sector lets (psl_build); n_sectors == 0 and let_size > 0: the paper's Cartesian lets (psl_build_grid)."""
        self._W = np.ascontiguousarray(psr["W"], np.float64)
        p = psr_params_t(psr["n_ebin"], psr["n_ring"], psr["e_min"], psr["e_bin_width"], psr["ring_width"], psr["z_phsp"],
                         self._W.ctypes.data_as(C.POINTER(C.c_double)), (C.c_double * 3)(*psr["sigma_src"]),
                         (C.c_double * 3)(*psr["z_src"]), (C.c_int32 * 3)(*psr["particle_type"]))
        j = jaws_t(*(jaws[k] for k in ("x1", "x2", "y1", "y2", "z_jx", "z_jy", "sad")))
        self.h = C.c_void_p()
        if n_sectors == 0:
            _check(lib().psl_build_grid(C.byref(p), C.byref(j), float(let_size), C.byref(self.h)))
        else:
            _check(lib().psl_build(C.byref(p), C.byref(j), n_sectors, C.byref(self.h)))
        self.n_ebin, self.n_groups = psr["n_ebin"], 3 * psr["n_ebin"]

    def set_direction_model(self, stype: int, c=None, mu=None, sigma_a=None, sigma_b=None):
        """Eq. 6 / Eq. 7 direction model of one sub-source (arrays [n_ebin][n_ring][K]); c=None restores the focal model."""
        if c is None:
            _check(lib().psl_set_direction_model(self.h, stype, 0, None, None, None, None))
            return
        arrs = [np.ascontiguousarray(a, np.float64) for a in (c, mu, sigma_a, sigma_b)]
        assert all(a.shape == arrs[0].shape for a in arrs)
        _check(lib().psl_set_direction_model(self.h, stype, arrs[0].shape[-1], *[a.ctypes.data_as(C.c_void_p) for a in arrs]))

    def __del__(self):
        if getattr(self, "h", None) and _lib is not None:
            _lib.psl_free(self.h)
            self.h = None

    def export(self) -> dict:
        n = C.c_size_t(0)
        _check(lib().psl_export(self.h, None, C.byref(n)))
        buf = np.zeros(n.value, np.uint8)
        _check(lib().psl_export(self.h, buf.ctypes.data_as(C.c_void_p), C.byref(n)))
        o, groups = 8, []
        G = int(buf[:8].view(np.uint64)[0])
        pad8 = lambda b: (b + 7) & ~7
        for _ in range(G):
            stype, ebin = buf[o:o + 8].view(np.int32)
            cnt = int(buf[o + 8:o + 16].view(np.uint64)[0])
            Wg = float(buf[o + 16:o + 24].view(np.float64)[0])
            o += 24
            arrs = []
            for dt, sz in ((np.uint16, 2), (np.uint16, 2), (np.uint32, 4), (np.uint32, 4)):
                arrs.append(buf[o:o + sz * cnt].view(dt).copy())
                o += pad8(sz * cnt)
            groups.append(dict(stype=int(stype), ebin=int(ebin), W=Wg, ring=arrs[0], sector=arrs[1], thresh=arrs[2], alias=arrs[3]))
        rect = buf[o:o + 96].view(np.float64).reshape(3, 4).copy()
        return dict(groups=groups, rect=rect)

    def allocate(self, n_histories: int) -> np.ndarray:
        off = np.empty(self.n_groups + 1, np.uint64)
        _check(lib().psl_allocate(self.h, n_histories, off.ctypes.data_as(C.c_void_p)))
        return off

    def workspace_bytes(self, phantom: DevicePhantom, batch: int, host: bool = False) -> int:
        f = lib().mc_host_workspace_bytes if host else lib().mc_workspace_bytes
        return int(f(self.h, C.byref(phantom.c), batch))

    def sample_debug(self, beam: dict, n_histories: int, seed: int, first: int, count: int, stream=None):
        """Returns a torch float32 tensor (2, count, 4): plane 0 = (x,y,z,E), plane 1 = (u,v,w,status)."""
        import torch
        out = torch.empty((2, count, 4), dtype=torch.float32, device="cuda")
        _check(lib().mc_sample_debug(self.h, C.byref(_beam(beam)), first, count, n_histories, seed, out.data_ptr(),
                                     _stream_ptr(stream)))
        return out

    def dose(self, phantom: DevicePhantom, beam: dict, n_histories: int, seed: int, batch: int = DEFAULT_BATCH, dose_out=None,
             **opt):
        """mc_dose.  Returns dose_out (torch float64 on the device, MeV/g per history)."""
        import torch
        if dose_out is None and opt.get("dose_acc") is None:
            dose_out = torch.empty(phantom.nvox, dtype=torch.float64, device=phantom.device)
        if opt.get("workspace") is None:
            opt["workspace"] = workspace(self.workspace_bytes(phantom, batch), phantom.device)
        o = _opts(**opt)
        _check(lib().mc_dose(self.h, C.byref(phantom.c), C.byref(_beam(beam)), n_histories, seed, batch,
                             dose_out.data_ptr() if dose_out is not None else None, C.byref(o)))
        return dose_out

    def dose_static(self, phantom: DevicePhantom, beam: dict, n_histories: int, seed: int, batch: int = 1 << 14, dose_out=None,
                    **opt):
        """mc_dose_static: mc_dose on the library's static device scratch (no allocation inside the call; dose_out or
        dose_acc must be given by callers that want none in the binding either).  Same bits as dose()."""
        import torch
        if dose_out is None and opt.get("dose_acc") is None:
            dose_out = torch.empty(phantom.nvox, dtype=torch.float64, device=phantom.device)
        assert opt.get("workspace") is None, "dose_static takes no workspace"
        o = _opts(**opt)
        _check(lib().mc_dose_static(self.h, C.byref(phantom.c), C.byref(_beam(beam)), n_histories, seed, batch,
                                    dose_out.data_ptr() if dose_out is not None else None, C.byref(o)))
        return dose_out

    def dose_host(self, ph: dict, beam: dict, n_histories: int, seed: int, batch: int = DEFAULT_BATCH, dose_out: np.ndarray = None,
                  density: np.ndarray = None, material: np.ndarray = None, **opt) -> np.ndarray:
        """mc_dose_host: host phantom arrays in, host dose out (copies inside the call)."""
        density = np.ascontiguousarray(ph["density"], np.float32) if density is None else density
        material = np.ascontiguousarray(ph["material"], np.uint8) if material is None else material
        if dose_out is None:
            dose_out = np.empty(density.size, np.float64)
        c = _phantom_struct(ph, density.ctypes.data, material.ctypes.data)
        if opt.get("workspace") is None:
            opt["workspace"] = workspace(int(lib().mc_host_workspace_bytes(self.h, C.byref(c), batch)))
        o = _opts(**opt)
        _check(lib().mc_dose_host(self.h, C.byref(c), C.byref(_beam(beam)), n_histories, seed, batch,
                                  dose_out.ctypes.data_as(C.c_void_p), C.byref(o)))
        return dose_out


def transport_debug(phantom: DevicePhantom, ptype: int, soa, first: int, seed: int, dose_acc, **opt):
    """mc_transport_debug on a (2, count, 4) float32 device tensor in mc_sample_debug's layout."""
    count = soa.shape[1]
    if opt.get("workspace") is None:
        opt["workspace"] = workspace(int(lib().mc_workspace_bytes(None, C.byref(phantom.c), max(count, 1))), phantom.device)
    o = _opts(dose_acc=dose_acc, pipelines=1, **opt)
    _check(lib().mc_transport_debug(C.byref(phantom.c), ptype, soa.data_ptr(), first, count, seed, C.byref(o)))


def philox_debug(seed: int, history: int, track: int, block: int) -> np.ndarray:
    out = np.empty(4, np.uint32)
    _check(lib().mc_philox_debug(seed, history, track, block, out.ctypes.data_as(C.c_void_p)))
    return out


def xs_debug(rhomax, e_max: float, energies) -> np.ndarray:
    """k_photon's cross-section lookup for `energies` (MeV): rows of (sigma_KN, ln^2(E/1.022), mu_max)."""
    rm = np.ascontiguousarray(rhomax, np.float32)
    e = np.ascontiguousarray(energies, np.float32)
    out = np.empty((e.size, 3), np.float32)
    _check(lib().mc_xs_debug(rm.ctypes.data_as(C.c_void_p), float(e_max), e.ctypes.data_as(C.c_void_p), e.size, out.ctypes.data_as(C.c_void_p)))
    return out


def plan_allocate(psls, n_histories: int) -> np.ndarray:
    """Eq. 3 across the beams of a plan: histories per beam, proportional to each beam's active weight."""
    arr = (C.c_void_p * len(psls))(*[p.h for p in psls])
    out = np.zeros(len(psls), np.uint64)
    _check(lib().mc_plan_allocate(arr, len(psls), n_histories, out.ctypes.data_as(C.c_void_p)))
    return out


def plan_dose(psls, phantom, beams, n_histories: int, seed: int, batch: int = DEFAULT_BATCH, rank: int = 0, world: int = 1,
              dose_out=None, dose_acc=None, **opt):
    """mc_plan_dose: a multi-beam plan (PAPER.md:73-80 S1-S2) - Eq. 3 over all beams, beam i with seed + i, one int64 grid.
    With world > 1 this call runs shard `rank` of every beam's histories; the caller all-reduces the returned grid
    (int64, SUM: bit-exact).  Returns (acc int64 on the device, histories per beam)."""
    import torch
    if dose_acc is None:
        dose_acc = torch.zeros(phantom.nvox, dtype=torch.int64, device=phantom.device)
    if opt.get("workspace") is None:
        opt["workspace"] = workspace(int(lib().mc_workspace_bytes(None, C.byref(phantom.c), batch)), phantom.device)
    o = _opts(dose_acc=dose_acc, shard=(rank, world), **opt)
    arr = (C.c_void_p * len(psls))(*[p.h for p in psls])
    bm = (beam_geom_t * len(beams))(*[_beam(b) for b in beams])
    n_beam = np.zeros(len(psls), np.uint64)
    _check(lib().mc_plan_dose(arr, bm, len(psls), C.byref(phantom.c), n_histories, seed, batch,
                              dose_out.data_ptr() if dose_out is not None else None, C.byref(o), n_beam.ctypes.data_as(C.c_void_p)))
    return dose_acc, n_beam


def shard_range(n_histories: int, rank: int, world: int) -> tuple[int, int]:
    """Contiguous history-id range of one rank (multi-GPU: histories are independent)."""
    return n_histories * rank // world, n_histories * (rank + 1) // world
