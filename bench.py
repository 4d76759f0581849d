#!/usr/bin/env python
"""bench.py — primary histories/s of the whole hot path (k_sample → k_photon/k_electron → scoring → finalise).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config C4] [--batch B]

Headline workload: BASELINE.json configs[4] (C4: 256^3 water at 0.2 cm, 40x40 cm field, 48x64x32 lets, its full 1e9
histories) — the metric names no configuration, so the largest single-GPU workload carries it.  One "step" = one mc_dose
pass over the whole workload.  The other configurations (C1, C2, C3 as a 7-beam plan through mc_plan_dose) are timed in
the same run and reported under `all_configs`.  N > 1 (torchrun, one rank per GPU): weak scaling — every rank runs the
config's histories as its contiguous id range of an N-times larger allocation, then one int64 all-reduce of the dose
grid (the path's only exchange; bit-exact because the tally is integer).  Prints ONE JSON line on rank 0.
`--impl reference` times the CPU oracle (oracle/) on the host cores.
"""
from __future__ import annotations

import argparse
import json
import multiprocessing as mp
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "primary histories/sec per B200 (sampling+transport+scoring); warp exec eff."
UNIT = "histories/s"
ALU_LANES = 148 * 128                     # 148 SMs x 4 schedulers x 32 lanes issue one thread-instruction per clock

# Algorithmic work of one event, in thread-instructions (DESIGN.md §5 derives each line; written down ONCE, not measured
# on the kernels).  Multiplied by the oracle's event counts per history this is the numerator of the ALU roofline.
BUDGET = {"sample": 300.0,      # per history: 2 Philox blocks (2 x 40), alias pick, position, energy, source point, direction, jaw, transform, entry, compaction
          "track": 30.0,        # per transported track: load, stream set-up, voxel index
          "flight": 130.0,      # Philox block 40, cross-section lookup 30, log + division 12, move + locate + gather 30, selection 18
          "kahn_trial": 70.0,   # Philox block 40, trial 30
          "scatter": 60.0,      # accepted Compton: kinematics 10, rotation 30, recoil direction + child id + queue push 20
          "pair": 60.0,         # split, two charged children, isotropic direction, two annihilation photons
          "substep": 60.0,      # gather 6, stopping power 6, step length 16, deposit 8, move + re-home 18, bounds 6
          "deflection": 90.0}   # Philox block 40, Highland angle 12, sincos + rotation 34, reciprocals 4
# SASS thread-instructions the kernels as built retire per history (ncu smsp__thread_inst_executed.sum / histories): side
# information, so that retired / algorithmic is visible.  Source: profiles/r2_launches.md (ncu launch lists of the end-of-round code).
RETIRED = {"C4": {"sample": 548, "photon": 3442, "electron": 3062}, "C1": {"sample": 471, "photon": 717, "electron": 874}}
# DRAM bytes (read + write) per history of each kernel class, from the `ncu --set full` captures in profiles/r2_top_kernels.md
NCU_DRAM_BYTES_PER_HISTORY = {"C4": {"sample": 27.8, "photon": 257.5, "electron": 177.8}, "C1": {"sample": 14.2, "photon": 34.6, "electron": 20.0}}


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default="C4")
    ap.add_argument("--batch", type=int, default=1 << 24)
    ap.add_argument("--histories", type=int, default=0, help="override histories per GPU (default: the config's)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-all-configs", action="store_true", help="time the headline workload only")
    ap.add_argument("--order", default="sorted", choices=["sorted", "mixed"])
    ap.add_argument("--static-lanes", action="store_true")
    ap.add_argument("--tile-sort", default="off", choices=["on", "off"], help="ablation: order every batch by entry tile (MC_FLAG_TILE_SORT)")
    ap.add_argument("--pipelines", type=int, default=0, help="0 = three overlapping launch sequences (the library default), 1 = serial")
    return ap.parse_args()


def describe(name: str) -> str:
    return {"C0": "32^3 water @0.5cm, 4x4 field, 8x16x8 lets", "C1": "64^3 water @0.25cm, 10x10 field, 24x32x16 lets, SSD 100",
            "C2": "128^3 slab phantom @0.25cm, 5x5 field", "C3": "256x256x120 patient-shaped, 8x8 field, 7-beam plan (mc_plan_dose)",
            "C4": "256^3 water @0.2cm, 40x40 field, 48x64x32 lets"}[name]


# ------------------------------------------------------------------ the oracle legs (CPU)
def oracle_sample_ranges(n_total: int, n_sample: int, pieces: int):
    """A bounded sample of the workload that keeps its type/energy mix: `pieces` equally spaced id ranges."""
    per = max(1, n_sample // pieces)
    return [(int(i * n_total / pieces), min(n_total, int(i * n_total / pieces) + per)) for i in range(pieces)]


def _oracle_run(name: str, n_total: int, ranges, beam_index: int = 0):
    """The oracle as it stands, single thread, over `ranges` of one beam.  Returns (histories, seconds, event counts)."""
    import numpy as np
    import oracle
    from paper_1503_01725_b200 import workloads
    cfg = workloads.make_config(name)
    opsl = oracle.Psl(cfg["psr"], cfg["jaws"], cfg["n_sectors"])
    oph = oracle.Phantom(cfg["phantom"])
    acc = np.zeros(oph.nvox, np.int64)
    done, counts = 0, {}
    t0 = time.perf_counter()
    for a, b in ranges:
        _, res, _ = opsl.dose(oph, cfg["beams"][beam_index], n_total, cfg["seed"] + beam_index, h_begin=a, h_end=b, acc=acc)
        done += b - a
        for k, v in res.items():
            if isinstance(v, int):
                counts[k] = counts.get(k, 0) + v
        counts["n_photon_primaries"] = counts.get("n_photon_primaries", 0) + res["n_hist"][0] + res["n_hist"][1]
    return done, time.perf_counter() - t0, counts


def _oracle_worker(args):
    return _oracle_run(*args)


def time_oracle(name: str, n_total: int, n_sample: int, procs: int = 1):
    """1 process: (rate, histories, seconds, counts).  procs > 1: the P-process aggregate over disjoint ranges."""
    pieces = 64 if name in ("C0", "C1", "C2") else 16            # every call re-scans the phantom: fewer pieces on the big ones
    ranges = oracle_sample_ranges(n_total, n_sample, pieces)
    if procs <= 1:
        done, dt, counts = _oracle_run(name, n_total, ranges)
        return done / dt, done, dt, counts
    chunks = [ranges[i::procs] for i in range(procs)]
    t0 = time.perf_counter()
    with mp.get_context("spawn").Pool(procs) as pool:
        out = pool.map(_oracle_worker, [(name, n_total, c) for c in chunks if c])
    wall = time.perf_counter() - t0
    done = sum(o[0] for o in out)
    busy = max(o[1] for o in out)                                 # the slowest process's own compute time (excludes interpreter start-up)
    return done / busy, done, wall, None


def algorithmic_work(counts: dict, histories: int) -> dict:
    """Thread-instructions per history of each kernel class = the oracle's event counts x BUDGET."""
    h = float(histories)
    photon_tracks = counts["n_photon_primaries"] - counts["n_jaw_rejected"] + counts["n_sec_photons"]
    ph = (BUDGET["track"] * max(photon_tracks, 0) + BUDGET["flight"] * counts["n_flights"] + BUDGET["kahn_trial"] * counts["n_kahn_trials"] +
          BUDGET["scatter"] * counts["n_compton"] + BUDGET["pair"] * counts["n_pair"]) / h
    el = (BUDGET["track"] * counts["n_electron_tracks"] + BUDGET["substep"] * counts["n_electron_steps"] +
          BUDGET["deflection"] * counts["n_deflections"]) / h
    ev = {k: counts[k] / h for k in ("n_flights", "n_kahn_trials", "n_compton", "n_pair", "n_electron_tracks", "n_electron_steps",
                                     "n_deflections", "n_deposits", "n_jaw_rejected")}
    return {"sample": BUDGET["sample"], "photon": ph, "electron": el, "events_per_history": ev}


def config_histories(name: str, cfg: dict) -> int:
    """Histories of one step: the config's count (C3: per beam x 7 beams, one plan)."""
    return cfg["n_histories"] * (len(cfg["beams"]) if name == "C3" else 1)


def run_reference(args):
    """The reference arm = the oracle as it stands on the host cores (single thread), on a bounded sample per step."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    from paper_1503_01725_b200 import workloads
    import oracle
    oracle.build()
    cfg = workloads.make_config(args.config, with_phantom=False)
    n_total = args.histories or cfg["n_histories"]
    n_sample = min(n_total, 2_000_000)
    for _ in range(args.warmup):
        time_oracle(args.config, n_total, min(n_sample, 50_000))
    rates, ms = [], []
    for _ in range(args.steps):
        r, done, dt, _ = time_oracle(args.config, n_total, n_sample)
        rates.append(r)
        ms.append(dt * 1e3)
    value = sum(rates) / len(rates)
    sample = "%d of %d histories per step, equally spaced id ranges (keeps the type/energy mix), beam 0" % (n_sample, n_total)
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": sum(ms) / len(ms), "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": "%s: %s" % (args.config, describe(args.config)), "histories_per_gpu": n_total},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample, "host_cores": os.cpu_count()},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


# ------------------------------------------------------------------ clocks during the timed region
class ClockSampler:
    Q = "clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown," \
        "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"

    def __init__(self, index: int):
        self.rows, self.p = [], None
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(index), "--query-gpu=" + self.Q, "--format=csv,noheader,nounits",
                                       "-lms", "100"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except OSError:
            self.p = None

    def _read(self):
        for line in self.p.stdout:
            self.rows.append((time.perf_counter(), [x.strip() for x in line.split(",")]))

    def stop(self, t0: float, t1: float) -> dict:
        if self.p is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.p.terminate()
        rows = [r for t, r in self.rows if t0 <= t <= t1] or [r for _, r in self.rows[-3:]]
        sm = sorted(int(r[0]) for r in rows if r[0].isdigit())
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        reasons = sorted({n for r in rows for n, v in zip(names, r[2:6]) if v.lower().startswith("active")})
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": int(rows[0][1]) if rows and rows[0][1].isdigit() else None,
                "reasons": reasons, "samples": len(rows)}


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return float(d["hbm_gbs"]), float(d.get("sm_max_mhz", 1965.0)), "measured (MEASURED_PEAKS.json)"
    return 6650.0, 1965.0, "fallback (B200_PROFILING.md)"


# ------------------------------------------------------------------ our arm (GPU)
class Workload:
    """One configuration resident in HBM, with the closures that run one step of it."""

    def __init__(self, name, args, B, workloads, world, rank):
        import torch
        self.name, self.B, self.args, self.world, self.rank = name, B, args, world, rank
        cfg = self.cfg = workloads.make_config(name)
        self.plan = name == "C3"                                   # seven beams, one int64 grid, Eq. 3 across beams
        per_gpu = (args.histories if (args.histories and name == args.config) else config_histories(name, cfg))
        self.per_gpu, self.n_total = per_gpu, per_gpu * world
        self.psl = B.Psl(cfg["psr"], cfg["jaws"], cfg["n_sectors"])
        self.ph = B.DevicePhantom(cfg["phantom"])
        nv = self.ph.nvox
        self.acc = torch.zeros(nv, dtype=torch.int64, device="cuda")
        self.dose = torch.empty(nv, dtype=torch.float64, device="cuda")
        self.ws = B.workspace(self.psl.workspace_bytes(self.ph, args.batch, host=True))
        self.order = B.MC_ORDER_MIXED if args.order == "mixed" else B.MC_ORDER_SORTED
        self.flags = (B.MC_FLAG_STATIC_LANES if args.static_lanes else 0) | \
            {"on": B.MC_FLAG_TILE_SORT, "off": 0}[args.tile_sort]
        self.hb, self.he = B.shard_range(self.n_total, rank, world)
        self.stream = torch.cuda.current_stream()

    def step(self, pipelines=None, timing=False):
        """One pass of the whole path.  timing: per-kernel-class CUDA events inside the library (the serial pass only)."""
        B, a = self.B, self.args
        pipelines = a.pipelines if pipelines is None else pipelines
        flags = self.flags | (B.MC_FLAG_TIMING if timing else 0)
        self.acc.zero_()
        if self.plan:
            nb = len(self.cfg["beams"])
            B.plan_dose([self.psl] * nb, self.ph, self.cfg["beams"], self.n_total, self.cfg["seed"], batch=a.batch, rank=self.rank,
                        world=self.world, dose_out=self.dose, dose_acc=self.acc, workspace=self.ws, flags=flags,
                        stream=self.stream, pipelines=pipelines)
        else:
            self.psl.dose(self.ph, self.cfg["beams"][0], self.n_total, self.cfg["seed"], batch=a.batch, dose_out=self.dose,
                          dose_acc=self.acc, workspace=self.ws, order=self.order, flags=flags, history_begin=self.hb,
                          history_end=self.he, stream=self.stream, pipelines=pipelines)

    def make_e2e(self):
        """End to end with HOST buffers (pinned): phantom up, dose down, inside the timed region."""
        import numpy as np
        import torch
        cfg, B, a = self.cfg, self.B, self.args
        hd = torch.from_numpy(np.ascontiguousarray(cfg["phantom"]["density"], np.float32)).pin_memory()
        hm = torch.from_numpy(np.ascontiguousarray(cfg["phantom"]["material"], np.uint8)).pin_memory()
        hout = torch.empty(self.ph.nvox, dtype=torch.float64).pin_memory()
        if self.plan:                                              # no host entry point at plan level: torch does the copies
            def run():
                self.ph.density.copy_(hd, non_blocking=True)
                self.ph.material.copy_(hm, non_blocking=True)
                self.step()
                hout.copy_(self.dose, non_blocking=True)
                torch.cuda.current_stream().synchronize()
        else:
            def run():
                self.psl.dose_host(cfg["phantom"], cfg["beams"][0], self.n_total, cfg["seed"], batch=a.batch, dose_out=hout.numpy(),
                                   density=hd.numpy(), material=hm.numpy(), workspace=self.ws, order=self.order,
                                   flags=self.flags, history_begin=self.hb, history_end=self.he, stream=self.stream)
        return run, 5 * self.ph.nvox, 8 * self.ph.nvox


def measure(w: Workload, steps: int, warmup: int, flush, dist=None):
    """W warm-up steps, K timed steps (CUDA events on the launching stream, L2 flushed before each), then a serial pass
    for the per-kernel times, then the end-to-end pass.  Returns a dict; times are this rank's."""
    import torch
    B = w.B
    for _ in range(warmup):
        w.step()
    torch.cuda.synchronize()
    if dist is not None:
        dist.barrier()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    launches, comm_ms, st = 0, 0.0, None
    for e0, e1 in ev:
        flush.fill_(1)                                   # L2 flush between timed steps (outside the timed events)
        e0.record(w.stream)
        w.step()
        if dist is not None:
            c0, c1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            c0.record(w.stream)
            dist.all_reduce(w.acc, op=dist.ReduceOp.SUM)   # the one exchange: int64 dose grid over NVLink
            c1.record(w.stream)
        e1.record(w.stream)
        st = B.stats()                                   # mc_dose is synchronous w.r.t. its stream: st is final
        launches += sum(st["launches"].values())
        if dist is not None:
            torch.cuda.synchronize()
            comm_ms += c0.elapsed_time(c1)
    torch.cuda.synchronize()
    total_ms = sum(e0.elapsed_time(e1) for e0, e1 in ev)
    # per-kernel-class times: the same steps with strictly serial launches (with several pipelines the classes overlap)
    ms_class = {k: 0.0 for k in B.KERNEL_CLASSES}
    serial_ms = 0.0
    for _ in range(steps):
        flush.fill_(1)
        w.step(pipelines=1, timing=True)
        s1 = B.stats()
        serial_ms += s1["ms_total"]
        for k in ms_class:
            ms_class[k] += s1["ms"][k]
    torch.cuda.synchronize()
    run, h2d, d2h = w.make_e2e()
    run()
    e2e_ms = []
    for _ in range(steps):
        flush.fill_(1)
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        run()                                            # returns after the dose is back in host memory
        e2e_ms.append((time.perf_counter() - t0) * 1e3)
    return {"total_ms": total_ms, "steps": steps, "stats": st, "launches": launches, "comm_ms": comm_ms,
            "ms_class": {k: v / steps for k, v in ms_class.items()}, "serial_ms": serial_ms / steps,
            "e2e_ms": sum(e2e_ms) / len(e2e_ms), "h2d": h2d, "d2h": d2h}


def summarise(w: Workload, m: dict, total_ms_max: float, clocks, alg, peaks) -> dict:
    """histories/s, end to end, per-kernel times and the rooflines of one measured workload."""
    hbm_peak, sm_max, which = peaks
    steps = m["steps"]
    value = w.n_total * steps / (total_ms_max * 1e-3)
    hist_rank = w.per_gpu                                   # histories this rank ran per step
    st, msc = m["stats"], m["ms_class"]
    out = {"workload": "%s: %s" % (w.name, describe(w.name)), "histories_per_step": w.n_total, "value": value, "unit": UNIT,
           "ms_per_step": total_ms_max / steps,
           "e2e": {"value": w.n_total / (m["e2e_ms"] * 1e-3), "unit": UNIT, "h2d_bytes_per_step": m["h2d"], "d2h_bytes_per_step": m["d2h"],
                   "ms_per_step": m["e2e_ms"]},
           "gpu_launches_per_step": m["launches"] // steps,
           "kernel_ms_per_step": msc, "serial_ms_per_step": m["serial_ms"]}
    n_acc = hist_rank - st["n_jaw_rejected"]
    sample_gbs = 32.0 * n_acc / (msc["sample"] * 1e-3) / 1e9 if msc["sample"] > 0 else 0.0
    out["k_sample"] = {"achieved_GBps_survivors": sample_gbs, "frac_of_hbm_survivors": sample_gbs / hbm_peak,
                       "achieved_GBps_all_histories": 32.0 * hist_rank / (msc["sample"] * 1e-3) / 1e9 if msc["sample"] > 0 else 0.0,
                       "histories_per_s": hist_rank / (msc["sample"] * 1e-3) if msc["sample"] > 0 else None}
    out["k_sample"]["frac_of_hbm_all_histories"] = out["k_sample"]["achieved_GBps_all_histories"] / hbm_peak
    if alg is not None:
        f_clk = ((clocks or {}).get("sm_mhz") or sm_max) * 1e6
        peak = ALU_LANES * f_clk / 1e12                      # T thread-instr/s at the SM clock seen under load
        dom = max(("sample", "photon", "electron"), key=lambda k: msc[k])
        ach = {k: alg[k] * hist_rank / (msc[k] * 1e-3) / 1e12 if msc[k] > 0 else 0.0 for k in ("sample", "photon", "electron")}
        retired = RETIRED.get(w.name, {})
        out["roofline"] = {"bound": "alu", "kernel": "k_" + dom, "achieved": ach[dom], "peak": peak, "unit": "Tinst/s (thread)",
                           "frac": ach[dom] / peak, "traffic": (NCU_DRAM_BYTES_PER_HISTORY.get(w.name, {}).get(dom) or 0) * hist_rank or None,
                           "peak_source": "148 SM x 128 lanes x SM clock under load (DESIGN.md §5)",
                           "alg_thread_inst_per_history": alg[dom], "alg_source": "oracle event counts x BUDGET (bench.py, DESIGN.md §5)",
                           "retired_thread_inst_per_history": retired.get(dom),
                           "per_kernel_frac": {k: ach[k] / peak for k in ach}}
        whole = (alg["sample"] + alg["photon"] + alg["electron"]) * hist_rank / (m["serial_ms"] * 1e-3) / 1e12 / peak
        out["whole_path_alu_frac"] = whole
        out["alg_thread_inst_per_history"] = {k: alg[k] for k in ("sample", "photon", "electron")}
        out["events_per_history"] = alg["events_per_history"]
    return out


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_1503_01725_b200 import binding as B, workloads

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    B.lib()                                              # fails loudly if libpslmc.so is missing
    D = dist if world > 1 else None
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")       # > 126 MB L2
    peaks = load_peaks()
    warmup = max(args.warmup, 3)

    def max_over_ranks(x: float) -> float:
        t = torch.tensor([x], dtype=torch.float64, device="cuda")
        if world > 1:
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
        return float(t.item())

    # ---- the headline workload
    head = Workload(args.config, args, B, workloads, world, rank)
    clocks = ClockSampler(local) if rank == 0 else None
    t_begin = time.perf_counter()
    m = measure(head, args.steps, warmup, flush, D)
    t_end = time.perf_counter()
    total_ms = max_over_ranks(m["total_ms"])
    ck = clocks.stop(t_begin, t_end) if clocks else None

    # ---- multi-GPU self-check (outside the timed region): the all-reduced int64 grid of a sharded C1 run must equal a
    # single-rank run of the same allocation bit for bit, ledgers included
    selfcheck = None
    if world > 1:
        c1 = workloads.make_config("C1")
        p1, ph1 = B.Psl(c1["psr"], c1["jaws"], c1["n_sectors"]), B.DevicePhantom(c1["phantom"])
        n1 = 2_000_000 * world
        hb, he = B.shard_range(n1, rank, world)
        a1 = torch.zeros(ph1.nvox, dtype=torch.int64, device="cuda")
        p1.dose(ph1, c1["beams"][0], n1, c1["seed"], batch=1 << 20, dose_acc=a1, history_begin=hb, history_end=he)
        led = torch.tensor([B.stats()["ledger"][k] for k in B.LEDGERS], dtype=torch.int64, device="cuda")
        dist.all_reduce(a1, op=dist.ReduceOp.SUM)
        dist.all_reduce(led, op=dist.ReduceOp.SUM)
        if rank == 0:
            a0 = torch.zeros_like(a1)
            p1.dose(ph1, c1["beams"][0], n1, c1["seed"], batch=1 << 21, dose_acc=a0)
            L0 = B.stats()["ledger"]
            selfcheck = {"workload": "C1, %d histories over %d ranks vs one rank" % (n1, world), "grid_bit_exact": bool(torch.equal(a0, a1)),
                         "ledgers_exact": led.tolist() == [L0[k] for k in B.LEDGERS]}

    # ---- the other configurations (single GPU runs only: they explain the headline, they are not scaled)
    others = {}
    if not args.no_all_configs and world == 1:
        for name in ("C1", "C2", "C3", "C4"):
            if name == args.config:
                continue
            w = Workload(name, args, B, workloads, world, rank)
            others[name] = (w, measure(w, 3, 3, flush, None))
            del w
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return
    finish(args, B, head, m, total_ms, ck, others, selfcheck, peaks, world, warmup)
    if world > 1:
        dist.destroy_process_group()


def cpu_baseline(name: str, n_total: int, budget_s: float, with_p: bool):
    """The oracle as it stands on the host cores: 1 process on a bounded sample (also the source of the event counts), and
    optionally the aggregate of one single-threaded process per core over disjoint ranges."""
    probe_rate, _, _, _ = time_oracle(name, n_total, 20_000)                  # sizes the sample to the time budget
    n_sample = int(min(n_total, max(50_000, probe_rate * budget_s)))
    v, done, dt, counts = time_oracle(name, n_total, n_sample)
    out = {"value": v, "unit": UNIT, "cores": 1, "kind": "oracle", "host_cores": os.cpu_count(),
           "sample": "%d of %d histories in equally spaced id ranges (beam 0), %.1f s, single thread" % (done, n_total, dt)}
    if with_p:
        procs = max(1, os.cpu_count() or 1)
        vp, donep, wall, _ = time_oracle(name, n_total, int(min(n_total, n_sample * min(procs, 8))), procs=procs)
        out["p_process"] = {"processes": procs, "value": vp, "unit": UNIT,
                            "sample": "%d histories over %d single-threaded oracle processes, %.1f s wall" % (donep, procs, wall)}
    return out, counts, done


def finish(args, B, head, m, total_ms, ck, others, selfcheck, peaks, world, warmup):
    from paper_1503_01725_b200 import probes
    cfg_n = config_histories(head.name, head.cfg) // (len(head.cfg["beams"]) if head.plan else 1)
    alg, base = None, None
    if not args.no_cpu_baseline:
        base, counts, done = cpu_baseline(head.name, cfg_n, 12.0, with_p=(world == 1))
        alg = algorithmic_work(counts, done)
    out = summarise(head, m, total_ms, ck, alg, peaks)
    line = {"metric": METRIC, "value": out["value"], "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": warmup,
            "ms_per_step": out["ms_per_step"], "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32", "data": "synthetic",
            "config": {"workload": out["workload"], "histories_per_gpu": head.per_gpu, "seed": head.cfg["seed"], "batch": args.batch,
                       "order": args.order, "lane_refill": not args.static_lanes, "tile_sort": args.tile_sort, "pipelines": args.pipelines or 3,
                       "parallelism": "history-range shards x%d + int64 all-reduce" % world if world > 1 else "single GPU",
                       "l2": "flushed between timed steps (256 MiB write)"},
            "clocks": ck, "e2e": out["e2e"], "gpu_launches": m["launches"]}
    for k in ("roofline", "whole_path_alu_frac", "alg_thread_inst_per_history", "events_per_history", "kernel_ms_per_step", "serial_ms_per_step", "k_sample"):
        if k in out:
            line[k] = out[k]
    line["kernel_ms_note"] = "serial pass (pipelines=1); the timed region overlaps three pipelines"
    if base is not None:
        line["cpu_baseline"] = base
    # the random-access ceilings of this phantom (probes): gathers from the packed phantom, int64 REDs into the grid
    try:
        nv = head.ph.nvox
        g_rate, r_rate = probes.gather32_rate(nv, 1 << 27), probes.red64_rate(nv, 1 << 27)
        ra = {"gather32_ceiling_per_s": g_rate, "red64_ceiling_per_s": r_rate, "footprint_bytes": 12 * nv}
        if alg is not None:
            ev = alg["events_per_history"]
            gathers, reds = ev["n_flights"] + ev["n_electron_steps"], ev["n_deposits"]
            ceil = 1.0 / (gathers / g_rate + reds / r_rate)       # histories/s if nothing but these accesses ran, one after the other
            ra.update({"gathers_per_history": gathers, "deposits_per_history": reds, "ceiling_histories_per_s": ceil,
                       "frac": head.per_gpu / (m["serial_ms"] * 1e-3) / ceil})
        line["random_access"] = ra
    except (ImportError, RuntimeError, OSError) as e:
        line["random_access"] = {"unavailable": str(e)}
    if world > 1:
        nbytes = 8 * head.ph.nvox
        line["comm"] = {"all_reduce_bytes": nbytes, "all_reduce_ms_per_step": m["comm_ms"] / args.steps,
                        "compute_ms_per_step": out["ms_per_step"] - m["comm_ms"] / args.steps, "self_check": selfcheck}
    if others:
        allc = {head.name: {k: out[k] for k in ("workload", "histories_per_step", "value", "ms_per_step", "e2e", "gpu_launches_per_step", "kernel_ms_per_step")}}
        for name, (w, mm) in others.items():
            n1 = config_histories(name, w.cfg) // (len(w.cfg["beams"]) if w.plan else 1)
            a1, b1 = None, None
            if not args.no_cpu_baseline:
                b1, c1, d1 = cpu_baseline(name, n1, 4.0, with_p=False)
                a1 = algorithmic_work(c1, d1)
            o = summarise(w, mm, mm["total_ms"], ck, a1, peaks)
            o["steps"], o["warmup"] = 3, 3
            if b1 is not None:
                o["cpu_baseline"] = b1
            allc[name] = o
        line["all_configs"] = allc
    line["paper_context"] = "Table 1 (unstated GPU, OpenCL): 1e9 particles, 40x40 cm2 water: 111.81 s = 0.89e7 histories/s; 10x10: 69.15 s"

    def clean(x):                                        # strict JSON: no NaN
        if isinstance(x, dict):
            return {k: clean(v) for k, v in x.items()}
        if isinstance(x, float) and x != x:
            return None
        return x
    print(json.dumps(clean(line)))


if __name__ == "__main__":
    a = parse()
    if a.impl == "reference":
        run_reference(a)
    else:
        run_ours(a)
