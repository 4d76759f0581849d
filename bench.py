#!/usr/bin/env python
"""bench.py — primary histories/s of the whole hot path (k_sample → k_photon/k_electron → scoring →
finalise) on BASELINE.json configs[1] (C1: 64^3 water at 0.25 cm, 10x10 cm field, 1e7 histories, seed 2).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config C1] [--batch B]

One "step" = one mc_dose pass over the workload.  N > 1 (torchrun, one rank per GPU): weak scaling —
every rank runs 1e7 histories (its contiguous id range of an N*1e7-history allocation), then one
int64 all-reduce of the dose grid (the path's only exchange; bit-exact because the tally is integer).
Prints ONE JSON line on rank 0.  `--impl reference` times the CPU oracle (oracle/) on the host cores.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "primary histories/sec per B200 (sampling+transport+scoring)"
UNIT = "histories/s"
# thread-instructions per C1 history of the transport kernels (ncu
# smsp__thread_inst_executed.sum / histories, profiles/), and the issue peak 148 SM x 128 lanes x f.
ALU_LANES = 148 * 128


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default="C1")
    ap.add_argument("--batch", type=int, default=1 << 22)
    ap.add_argument("--histories", type=int, default=0, help="override histories per GPU (default: the config's)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--order", default="sorted", choices=["sorted", "mixed"])
    ap.add_argument("--static-lanes", action="store_true")
    ap.add_argument("--pipelines", type=int, default=0, help="0 = library default (2 overlapping launch sequences), 1 = serial")
    return ap.parse_args()


# ------------------------------------------------------------------ the oracle legs (CPU)
def oracle_sample_ranges(n_total: int, n_sample: int, pieces: int = 64):
    """A bounded sample of the workload that keeps its type/energy mix: `pieces` equally spaced id ranges."""
    per = max(1, n_sample // pieces)
    return [(int(i * n_total / pieces), min(n_total, int(i * n_total / pieces) + per)) for i in range(pieces)]


def time_oracle(cfg, n_total: int, n_sample: int):
    import oracle
    opsl = oracle.Psl(cfg["psr"], cfg["jaws"], cfg["n_sectors"])
    oph = oracle.Phantom(cfg["phantom"])
    import numpy as np
    acc = np.zeros(oph.nvox, np.int64)
    done = 0
    t0 = time.perf_counter()
    for a, b in oracle_sample_ranges(n_total, n_sample):
        opsl.dose(oph, cfg["beams"][0], n_total, cfg["seed"], h_begin=a, h_end=b, acc=acc)
        done += b - a
    dt = time.perf_counter() - t0
    return done / dt, done, dt


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from paper_1503_01725_b200 import workloads
    import oracle
    oracle.build()
    cfg = workloads.make_config(args.config)
    n_total = args.histories or cfg["n_histories"]
    n_sample = min(n_total, 4_000_000)
    for _ in range(args.warmup):
        time_oracle(cfg, n_total, min(n_sample, 100_000))
    rates, ms = [], []
    for _ in range(args.steps):
        r, done, dt = time_oracle(cfg, n_total, n_sample)
        rates.append(done / dt)
        ms.append(dt * 1e3)
    value = sum(rates) / len(rates)
    sample = "%d of %d histories per step: 64 equally spaced id ranges (keeps the type/energy mix)" % (n_sample, n_total)
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": sum(ms) / len(ms), "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": "%s: %s" % (args.config, describe(args.config)), "histories": n_total},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


def describe(name: str) -> str:
    return {"C0": "32^3 water @0.5cm, 4x4 field, 8x16x8 lets", "C1": "64^3 water @0.25cm, 10x10 field, 24x32x16 lets, SSD 100",
            "C2": "128^3 slab phantom @0.25cm, 5x5 field", "C3": "256x256x120 patient-shaped, 8x8 field, beam 0",
            "C4": "256^3 water @0.2cm, 40x40 field, 48x64x32 lets"}[name]


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


# ------------------------------------------------------------------ our arm (GPU)
# Algorithmic work per history of the bench workload, stated in DESIGN.md §Roofline and measured once
# with ncu (profiles/): SASS thread-instructions the transport kernels retire per C1 primary history,
# and the bytes k_sample must write per history (32 B per particle that passes the jaws).
ALG_THREAD_INST_PER_HISTORY = {"C1": {"photon": 677.0, "electron": 849.0, "sample": 507.0},      # profiles/r1c_launches.md
                               "C4": {"photon": 2575.0, "electron": 2604.0, "sample": 600.0}}    # profiles/r1b_ablation_c4.md (batch 2^22, sorted)
# DRAM bytes (read + write) per step of each kernel class, from the ncu --set full captures of profiles/r1c_top_kernels.md
# (the two primary-batch launches; the path's working set is L2-resident, so this is far below any HBM bound)
NCU_DRAM_BYTES_PER_STEP = {"C1": {"photon": 2.17e8, "electron": 1.42e8, "sample": 6.5e7}}
SAMPLE_BYTES_PER_PARTICLE = 32.0


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return float(d["hbm_gbs"]), float(d.get("sm_max_mhz", 1965.0)), "measured"
    return 6650.0, 1965.0, "fallback"


def run_ours(args):
    import numpy as np
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

    cfg = workloads.make_config(args.config)
    per_gpu = args.histories or cfg["n_histories"]
    n_total = per_gpu * world
    hb, he = B.shard_range(n_total, rank, world)
    psl = B.Psl(cfg["psr"], cfg["jaws"], cfg["n_sectors"])
    ph = B.DevicePhantom(cfg["phantom"])
    beam, seed = cfg["beams"][0], cfg["seed"]
    ws = torch.empty(psl.workspace_bytes(ph, args.batch), dtype=torch.uint8, device="cuda")
    acc = torch.zeros(ph.nvox, dtype=torch.int64, device="cuda")
    dose = torch.empty(ph.nvox, dtype=torch.float64, device="cuda")
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")       # > 126 MB L2
    order = B.MC_ORDER_MIXED if args.order == "mixed" else B.MC_ORDER_SORTED
    flags = B.MC_FLAG_TIMING | (B.MC_FLAG_STATIC_LANES if args.static_lanes else 0)
    stream = torch.cuda.current_stream()

    def step(pipelines=args.pipelines):
        acc.zero_()
        psl.dose(ph, beam, n_total, seed, batch=args.batch, dose_out=dose, dose_acc=acc, workspace=ws, order=order,
                 flags=flags, history_begin=hb, history_end=he, stream=stream, pipelines=pipelines)
        if world > 1:
            dist.all_reduce(acc, op=dist.ReduceOp.SUM)   # the one exchange: int64 dose grid over NVLink

    for _ in range(max(args.warmup, 3)):
        step()
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    clocks = ClockSampler(local) if rank == 0 else None
    t_begin = time.perf_counter()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    launches = 0
    for e0, e1 in ev:
        flush.fill_(1)                                   # L2 flush between timed steps (outside the timed events)
        e0.record(stream)
        step()
        e1.record(stream)
        st = B.stats()                                   # mc_dose is synchronous w.r.t. its stream: st is final
        launches += sum(st["launches"].values())
    torch.cuda.synchronize()
    # Per-kernel-class times for the roofline: the same K steps once more with strictly serial launches
    # (pipelines = 1), because with overlapping pipelines the classes share the GPU and their event times
    # are not disjoint.  `value` above is the overlapped run; these are the kernels' own durations.
    ms_class = {k: 0.0 for k in B.KERNEL_CLASSES}
    serial_ms = 0.0
    for _ in range(args.steps):
        flush.fill_(1)
        step(pipelines=1)
        st1 = B.stats()
        serial_ms += st1["ms_total"]
        for k in ms_class:
            ms_class[k] += st1["ms"][k]
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    t_end = time.perf_counter()
    ms_steps = [e0.elapsed_time(e1) for e0, e1 in ev]
    total_ms = torch.tensor([sum(ms_steps)], dtype=torch.float64, device="cuda")
    if world > 1:
        dist.all_reduce(total_ms, op=dist.ReduceOp.MAX)
    total_ms = float(total_ms.item())
    value = n_total * args.steps / (total_ms * 1e-3)
    ck = clocks.stop(t_begin, t_end) if clocks else None

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- end to end through the C ABI with HOST buffers (pinned), copies inside the timed region
    hd = torch.from_numpy(np.ascontiguousarray(cfg["phantom"]["density"], np.float32)).pin_memory()
    hm = torch.from_numpy(np.ascontiguousarray(cfg["phantom"]["material"], np.uint8)).pin_memory()
    hout = torch.empty(ph.nvox, dtype=torch.float64).pin_memory()
    def e2e_step():
        psl.dose_host(cfg["phantom"], beam, n_total, seed, batch=args.batch, dose_out=hout.numpy(), density=hd.numpy(),
                      material=hm.numpy(), workspace=ws, order=order, history_begin=hb, history_end=he, stream=stream)
    e2e_step()
    e2e_ms = []
    for _ in range(args.steps):
        flush.fill_(1)
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        e2e_step()                                       # returns after the dose is back in host memory
        e2e_ms.append((time.perf_counter() - t0) * 1e3)
    e2e_value = per_gpu * world / (sum(e2e_ms) / len(e2e_ms) * 1e-3)

    # ---- roofline of the dominant kernel class (live CUDA-event times of the timed region)
    hbm_peak, sm_max, which = load_peaks()
    dom = max(("sample", "photon", "electron"), key=lambda k: ms_class[k])
    hist_rank = (he - hb) * args.steps
    alg = ALG_THREAD_INST_PER_HISTORY.get(args.config)
    if alg is None:                                      # no ncu count for this workload: report times only
        alg = {"photon": float("nan"), "electron": float("nan"), "sample": float("nan")}
    n_acc = hist_rank - st["n_jaw_rejected"] * args.steps
    sample_gbs = SAMPLE_BYTES_PER_PARTICLE * n_acc / (ms_class["sample"] * 1e-3) / 1e9 if ms_class["sample"] > 0 else 0.0
    if dom == "sample":
        roof = {"bound": "hbm", "kernel": "k_sample", "achieved": sample_gbs, "peak": hbm_peak, "unit": "GB/s",
                "frac": sample_gbs / hbm_peak, "traffic": None, "peak_source": which}
    else:
        f_clk = (ck["sm_mhz"] or sm_max) * 1e6 if ck else sm_max * 1e6
        peak = ALU_LANES * f_clk / 1e12                  # T thread-instr/s at the SM clock seen under load
        achieved = alg[dom] * hist_rank / (ms_class[dom] * 1e-3) / 1e12
        roof = {"bound": "alu", "kernel": "k_" + dom, "achieved": achieved, "peak": peak, "unit": "Tinst/s (thread)",
                "frac": achieved / peak, "traffic": NCU_DRAM_BYTES_PER_STEP.get(args.config, {}).get(dom),
                "peak_source": "148 SM x 128 lanes x SM clock under load (DESIGN.md)", "alg_thread_inst_per_history": alg[dom]}
    # the three hot kernels together: useful thread-instructions of a step over the lane-issue slots of the whole step
    f_clk_all = (ck["sm_mhz"] or sm_max) * 1e6 if ck else sm_max * 1e6
    whole = sum(alg.values()) * hist_rank / (total_ms * 1e-3) / (ALU_LANES * f_clk_all)
    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
        "ms_per_step": total_ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32", "data": "synthetic",
        "config": {"workload": "%s: %s" % (args.config, describe(args.config)), "histories_per_gpu": per_gpu, "seed": seed,
                   "batch": args.batch, "order": args.order, "lane_refill": not args.static_lanes, "pipelines": args.pipelines or 2,
                   "parallelism": "history-range shards x%d + int64 all-reduce" % world if world > 1 else "single GPU",
                   "l2": "flushed between timed steps (256 MiB write)"},
        "clocks": ck,
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": 5 * ph.nvox, "d2h_bytes_per_step": 8 * ph.nvox,
                "ms_per_step": sum(e2e_ms) / len(e2e_ms)},
        "gpu_launches": launches,
        "roofline": roof,
        "whole_path_lane_issue_frac": whole,
        "kernel_ms_per_step": {k: v / args.steps for k, v in ms_class.items()},
        "kernel_ms_note": "serial pass (pipelines=1, %.3f ms per step); the timed region overlaps two pipelines" % (serial_ms / args.steps),
        "k_sample": {"achieved_GBps": sample_gbs, "frac_of_hbm": sample_gbs / hbm_peak,
                     "histories_per_s": hist_rank / (ms_class["sample"] * 1e-3) if ms_class["sample"] > 0 else None},
        "paper_context": "Table 1 (unstated GPU, OpenCL): 1e9 histories 10x10 water in 69.15 s = 1.45e7 histories/s",
    }
    if not args.no_cpu_baseline and world == 1:
        v, done, dt = time_oracle(cfg, n_total, min(n_total, 20_000_000))
        out["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": 1, "kind": "oracle",
                               "sample": "%d of %d histories in 64 equally spaced id ranges, %.1f s" % (done, n_total, dt)}
    def clean(x):                                        # strict JSON: no NaN
        if isinstance(x, dict):
            return {k: clean(v) for k, v in x.items()}
        if isinstance(x, float) and x != x:
            return None
        return x
    print(json.dumps(clean(out)))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    a = parse()
    if a.impl == "reference":
        run_reference(a)
    else:
        run_ours(a)
