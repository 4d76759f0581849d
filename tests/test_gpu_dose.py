"""Whole-path mc_dose parity with the oracle, determinism and edge cases (python -m pytest tests -m gpu)."""
import numpy as np
import pytest

from test_gpu_parity import B, gpsl, COUNTERS          # noqa: F401  (fixtures)

pytestmark = pytest.mark.gpu


def gpu_dose(B, psl, dph, beam, N, seed, batch, want_fp=True, **opt):
    import torch
    hb, he = opt.get("history_begin", 0), opt.get("history_end", 0) or N
    fp = torch.zeros(he - hb, dtype=torch.int64, device="cuda") if want_fp else None
    acc = torch.zeros(dph.nvox, dtype=torch.int64, device="cuda")
    dose = torch.empty(dph.nvox, dtype=torch.float64, device="cuda")
    psl.dose(dph, beam, N, seed, batch=batch, dose_out=dose, dose_acc=acc, fingerprints=fp, **opt)
    st = B.stats()
    return acc.cpu().numpy(), dose.cpu().numpy(), st, (fp.cpu().numpy().view(np.uint64) if want_fp else None)


def compare_with_oracle(B, orc, g, o, ph_dict, beam, N, seed, batch, min_same=0.999, dose_tol=5e-3, frac_vox=0.995):
    dph, oph = B.DevicePhantom(ph_dict), orc.Phantom(ph_dict)
    acc, dose, st, fp = gpu_dose(B, g, dph, beam, N, seed, batch, flags=B.MC_FLAG_STATS)
    oacc, ores, ofp = o.dose(oph, beam, N, seed, fingerprints=True)
    ref = orc.finalise(oph, oacc, N)
    same = float((fp == ofp).mean())
    assert same >= min_same, same
    # integer bookkeeping
    assert st["n_hist"] == ores["n_hist"]
    assert abs(st["n_jaw_rejected"] - ores["n_jaw_rejected"]) <= max(2, 1e-4 * N)
    for k in COUNTERS:
        assert abs(st[k] - ores[k]) <= max(3, 2e-3 * ores[k]), (k, st[k], ores[k])
    L, OL = st["ledger"], ores["ledger"]
    assert int(acc.sum()) == L["deposited"]
    assert abs(L["deposited"] + L["escaped"] + L["jaw"] - L["incident"]) <= 1e-5 * L["incident"]
    for k in OL:
        assert abs(L[k] - OL[k]) <= 1e-3 * OL["incident"], k
    # dose: 0.5 % of local dose in voxels above 10 % of Dmax
    big = ref > 0.1 * ref.max()
    err = np.abs(dose[big] - ref[big]) / ref[big]
    assert np.median(err) < 1e-4
    assert (err <= dose_tol).mean() >= frac_vox, (float((err <= dose_tol).mean()), float(err.max()))
    # finalise: dose_out is exactly the scaled accumulator
    rho = np.asarray(ph_dict["density"], np.float64)
    V = ph_dict["dx"] * ph_dict["dy"] * ph_dict["dz"]
    exp = np.where(rho > 0, acc / 2.0 ** 32 / (np.where(rho > 0, rho, 1) * V * N), 0.0)
    assert np.allclose(dose, exp, rtol=1e-14, atol=0)
    return same, float(err.max()), float((err <= dose_tol).mean())


def test_dose_parity_c0_full(B, orc, gpsl, opsl, cfg):
    c = cfg("C0")
    compare_with_oracle(B, orc, gpsl("C0"), opsl("C0"), c["phantom"], c["beams"][0], c["n_histories"], c["seed"], batch=1 << 14)


def test_dose_parity_c1(B, orc, gpsl, opsl, cfg):
    c = cfg("C1")
    compare_with_oracle(B, orc, gpsl("C1"), opsl("C1"), c["phantom"], c["beams"][0], 2_000_000, c["seed"], batch=1 << 18)


def test_dose_parity_c2_heterogeneous(B, orc, gpsl, opsl, cfg):
    c = cfg("C2")
    compare_with_oracle(B, orc, gpsl("C2"), opsl("C2"), c["phantom"], c["beams"][0], 1_000_000, c["seed"], batch=300_000)


def test_dose_parity_c3_rotated_beam(B, orc, opsl, cfg):
    c = cfg("C3")
    g = B.Psl(c["psr"], c["jaws"], c["n_sectors"])
    compare_with_oracle(B, orc, g, opsl("C3"), c["phantom"], c["beams"][2], 500_000, 42, batch=1 << 17, frac_vox=0.98)


def test_dose_parity_c4_large_field(B, orc, gpsl, opsl, cfg):
    c = cfg("C4")
    compare_with_oracle(B, orc, gpsl("C4"), opsl("C4"), c["phantom"], c["beams"][0], 1_000_000, c["seed"], batch=1 << 20, frac_vox=0.98)


# ---------------------------------------------------------------- determinism contract (bit-exact)
def test_bitwise_identity_under_batch_order_partition(B, gpsl, cfg):
    c = cfg("C0")
    dph = B.DevicePhantom(c["phantom"])
    g, beam, N, seed = gpsl("C0"), c["beams"][0], 100_000, 1
    ref_acc, ref_dose, ref_st, ref_fp = gpu_dose(B, g, dph, beam, N, seed, 1 << 16)
    for batch, opt in ((1000, {}), (33_333, {}), (1 << 20, {}), (1 << 13, dict(order=B.MC_ORDER_MIXED)),
                       (1 << 15, dict(flags=B.MC_FLAG_STATIC_LANES)), (1 << 15, dict(flags=B.MC_FLAG_STATS | B.MC_FLAG_TIMING)),
                       (1 << 14, dict(pipelines=1)), (1 << 12, dict(pipelines=2, flags=B.MC_FLAG_TIMING)), (1 << 12, dict(pipelines=3)),
                       (1 << 16, dict(flags=B.MC_FLAG_STAGE_SCORING)), (1 << 12, dict(flags=B.MC_FLAG_STAGE_SCORING | B.MC_FLAG_STATS, order=B.MC_ORDER_MIXED)),
                       (1 << 14, dict(flags=B.MC_FLAG_TILE_SORT)), (1 << 13, dict(flags=B.MC_FLAG_TILE_SORT | B.MC_FLAG_STATS, order=B.MC_ORDER_MIXED, pipelines=1))):
        acc, dose, st, fp = gpu_dose(B, g, dph, beam, N, seed, batch, **opt)
        assert np.array_equal(acc, ref_acc), (batch, opt)
        assert np.array_equal(dose, ref_dose) and np.array_equal(fp, ref_fp)
        assert st["ledger"] == ref_st["ledger"] and st["n_jaw_rejected"] == ref_st["n_jaw_rejected"]
    # partitions of the history range, accumulated into one int64 grid
    import torch
    acc = torch.zeros(dph.nvox, dtype=torch.int64, device="cuda")
    led = {k: 0 for k in ref_st["ledger"]}
    for a, b in ((60_000, 100_000), (0, 1), (1, 25_000), (25_000, 60_000)):
        g.dose(dph, beam, N, seed, batch=9000, dose_acc=acc, history_begin=a, history_end=b)
        for k in led:
            led[k] += B.stats()["ledger"][k]
    assert np.array_equal(acc.cpu().numpy(), ref_acc) and led == ref_st["ledger"]


def test_mixed_order_is_bitwise_equal_on_c4(B, gpsl, cfg):
    c = cfg("C4")
    dph = B.DevicePhantom(c["phantom"])
    a0, _, s0, _ = gpu_dose(B, gpsl("C4"), dph, c["beams"][0], 3_000_000, 5, 1 << 20, want_fp=False)
    a1, _, s1, _ = gpu_dose(B, gpsl("C4"), dph, c["beams"][0], 3_000_000, 5, 1 << 18, want_fp=False, order=B.MC_ORDER_MIXED)
    assert np.array_equal(a0, a1) and s0["ledger"] == s1["ledger"]


def test_multi_beam_accumulation_and_conservation_c3(B, cfg):
    import torch
    c = cfg("C3")
    g = B.Psl(c["psr"], c["jaws"], c["n_sectors"])
    dph = B.DevicePhantom(c["phantom"])
    acc = torch.zeros(dph.nvox, dtype=torch.int64, device="cuda")
    dep = 0
    for b, beam in enumerate(c["beams"]):
        g.dose(dph, beam, 300_000, c["seed"] + b, batch=1 << 17, dose_acc=acc)
        L = B.stats()["ledger"]
        assert abs(L["deposited"] + L["escaped"] + L["jaw"] - L["incident"]) <= 1e-5 * L["incident"]
        dep += L["deposited"]
        assert int(acc.sum().item()) == dep
    d = acc.cpu().numpy().reshape(120, 256, 256)
    assert d[50:70, 118:138, 118:138].mean() > 5 * d[50:70, :20, :20].mean()     # beams cross at the isocentre


# ---------------------------------------------------------------- edge cases and errors
def test_edge_cases(B, gpsl, cfg):
    import torch
    c = cfg("C0")
    dph = B.DevicePhantom(c["phantom"])
    g, beam = gpsl("C0"), c["beams"][0]
    d = g.dose(dph, beam, 1, 3, batch=1)                                           # a single history
    assert d.shape[0] == dph.nvox and torch.isfinite(d).all()
    acc = torch.zeros(dph.nvox, dtype=torch.int64, device="cuda")
    g.dose(dph, beam, 1000, 3, batch=64, dose_acc=acc, history_begin=500, history_end=500)      # empty range
    assert int(acc.abs().sum().item()) == 0 and B.stats()["ledger"]["incident"] == 0
    with pytest.raises(B.PslmcError):
        g.dose(dph, beam, 1000, 3, batch=0)
    with pytest.raises(B.PslmcError):
        g.dose(dph, beam, 1000, 3, batch=64, history_begin=10, history_end=2000)
    small = torch.empty(1024, dtype=torch.uint8, device="cuda")
    with pytest.raises(B.PslmcError) as e:
        g.dose(dph, beam, 1000, 3, batch=1 << 16, workspace=small)
    assert e.value.code == -3
    # the empty shard [0, 0) is empty, not "everything" (MC_FLAG_RANGE, set by the binding for explicit ranges)
    acc.zero_()
    g.dose(dph, beam, 1000, 3, batch=64, dose_acc=acc, history_begin=0, history_end=0)
    assert int(acc.abs().sum().item()) == 0 and B.stats()["ledger"]["incident"] == 0
    # no workspace at the C ABI: MC_E_WORKSPACE, nothing is allocated behind the caller's back
    import ctypes as C
    o = B.mc_opts_t(); o.cuda_stream = int(torch.cuda.current_stream().cuda_stream)
    d0 = torch.empty(dph.nvox, dtype=torch.float64, device="cuda")
    rc = B.lib().mc_dose(g.h, C.byref(dph.c), C.byref(B._beam(beam)), 1000, 3, 64, d0.data_ptr(), C.byref(o))
    assert rc == -3
    ws = torch.empty(g.workspace_bytes(dph, 1 << 12), dtype=torch.uint8, device="cuda")
    a = g.dose(dph, beam, 20_000, 3, batch=1 << 12, workspace=ws).clone()
    b = g.dose(dph, beam, 20_000, 3, batch=1 << 12)
    assert torch.equal(a, b)
    # a side stream
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        c2 = g.dose(dph, beam, 20_000, 3, batch=1 << 12, stream=s)
    assert torch.equal(a, c2)


def test_no_allocation_inside_mc_dose_and_voxel_overflow(B, gpsl, cfg):
    """no hidden allocation inside mc_dose (free device memory is the same before and after, with the
    caller's workspace and streams); a voxel accumulator that wraps past 2^63 quanta is reported as MC_E_OVERFLOW."""
    import torch
    c = cfg("C0")
    dph = B.DevicePhantom(c["phantom"])
    g, beam = gpsl("C0"), c["beams"][0]
    ws = torch.empty(g.workspace_bytes(dph, 1 << 14), dtype=torch.uint8, device="cuda")
    acc = torch.zeros(dph.nvox, dtype=torch.int64, device="cuda")
    dose = torch.empty(dph.nvox, dtype=torch.float64, device="cuda")
    B.aux_streams()
    g.dose(dph, beam, 50_000, 3, batch=1 << 14, dose_out=dose, dose_acc=acc, workspace=ws)        # module load, first-use costs
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    for pipes in (1, 2, 3):
        g.dose(dph, beam, 50_000, 3, batch=1 << 14, dose_out=dose, dose_acc=acc, workspace=ws, pipelines=pipes, flags=B.MC_FLAG_TIMING)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0
    # overflow: the hottest voxel starts 1000 quanta below 2^63
    acc.zero_()
    g.dose(dph, beam, 50_000, 3, batch=1 << 14, dose_acc=acc, workspace=ws)
    hot = int(acc.argmax().item())
    acc.zero_(); acc[hot] = (1 << 63) - 1000
    with pytest.raises(B.PslmcError) as e:
        g.dose(dph, beam, 50_000, 3, batch=1 << 14, dose_acc=acc, workspace=ws)
    assert e.value.code == -5 and "wrapped" in str(e.value)


def test_two_host_threads_two_handles(B, cfg):
    """no process-global scratch or streams - two host threads, each with its own psl_t, workspace and streams,
    run mc_dose at the same time and get the bits of the serial runs."""
    import threading
    import torch
    c = cfg("C0")
    dph = B.DevicePhantom(c["phantom"])
    beam = c["beams"][0]
    ref, out = {}, {}
    psls = [B.Psl(c["psr"], c["jaws"], c["n_sectors"]) for _ in range(2)]
    for t, g in enumerate(psls):
        ref[t] = g.dose(dph, beam, 200_000, 11 + t, batch=1 << 13).clone()

    def work(t):
        torch.cuda.set_device(0)
        s = torch.cuda.Stream()
        aux = (torch.cuda.Stream(), torch.cuda.Stream())
        ws = torch.empty(psls[t].workspace_bytes(dph, 1 << 13), dtype=torch.uint8, device="cuda")
        with torch.cuda.stream(s):
            for _ in range(3):
                out[t] = psls[t].dose(dph, beam, 200_000, 11 + t, batch=1 << 13, workspace=ws, stream=s, aux=aux).clone()
        s.synchronize()

    th = [threading.Thread(target=work, args=(t,)) for t in range(2)]
    [t.start() for t in th]; [t.join() for t in th]
    assert torch.equal(out[0], ref[0]) and torch.equal(out[1], ref[1])


def test_host_entry_point_matches_device_entry_point(B, gpsl, cfg):
    c = cfg("C0")
    dph = B.DevicePhantom(c["phantom"])
    d_dev = gpsl("C0").dose(dph, c["beams"][0], 50_000, 1, batch=1 << 14).cpu().numpy()
    d_host = gpsl("C0").dose_host(c["phantom"], c["beams"][0], 50_000, 1, batch=1 << 14)
    assert np.array_equal(d_dev, d_host)


def test_vacuum_and_queue_stats(B, orc, cfg, wl):
    """A phantom with a vacuum gap (rho = 0): parity still holds; queue high-water marks are reported."""
    c = cfg("C1", False)
    n = 32
    rho = np.ones((n, n, n), np.float32); mat = np.zeros((n, n, n), np.uint8)
    rho[8:12] = 0.0
    rho[12:16], mat[12:16] = 1.85, 2
    ph = dict(nx=n, ny=n, nz=n, dx=0.5, dy=0.5, dz=0.5, ox=-8.0, oy=-8.0, oz=0.0, density=rho.reshape(-1), material=mat.reshape(-1))
    g, o = B.Psl(c["psr"], c["jaws"], 16), orc.Psl(c["psr"], c["jaws"], 16)
    compare_with_oracle(B, orc, g, o, ph, c["beams"][0], 300_000, 8, batch=1 << 16, frac_vox=0.98)
    st = B.stats()
    assert 0 < st["queue_high_water"] < 4 * (1 << 16) and st["launches"]["photon"] > 0


# ---------------------------------------------------------------- plan level (NEXT-4)
def test_plan_allocation_eq3_and_sharded_plan(B, cfg):
    """Eq. 3 across beams: histories per beam proportional to the beam's active weight; a 7-beam plan
    sharded over two 'ranks' (history ranges of every beam) adds up to the single-rank plan bit for bit."""
    import torch
    c = cfg("C3")
    fields = (4.0, 8.0, 12.0)
    psls = [B.Psl(c["psr"], dict(c["jaws"], x1=-f / 2, x2=f / 2, y1=-f / 2, y2=f / 2), c["n_sectors"]) for f in fields]
    W = np.array([sum(g["W"] for g in p.export()["groups"]) for p in psls])
    N = 1_000_003
    n = B.plan_allocate(psls, N).astype(np.int64)
    assert n.sum() == N and np.all(np.abs(n - N * W / W.sum()) < 1) and n[0] < n[1] < n[2]
    # C3: seven coplanar beams, one jaw setting
    dph = B.DevicePhantom(c["phantom"])
    g = B.Psl(c["psr"], c["jaws"], c["n_sectors"])
    beams = c["beams"]
    dose = torch.empty(dph.nvox, dtype=torch.float64, device="cuda")
    acc, nb = B.plan_dose([g] * len(beams), dph, beams, 2_100_000, 40, batch=1 << 18, dose_out=dose)
    st = B.stats()
    assert nb.tolist() == [300_000] * 7 and sum(st["n_hist"]) == 2_100_000 and int(acc.sum().item()) == st["ledger"]["deposited"]
    parts = [B.plan_dose([g] * len(beams), dph, beams, 2_100_000, 40, batch=1 << 17, rank=r, world=2)[0] for r in range(2)]
    assert torch.equal(parts[0] + parts[1], acc)
    # mc_plan_dose = one mc_dose per beam (seed + beam index) into one grid, normalised by the plan's histories
    acc2 = torch.zeros_like(acc)
    for i, beam in enumerate(beams):
        g.dose(dph, beam, 300_000, 40 + i, batch=1 << 16, dose_acc=acc2)
    assert torch.equal(acc, acc2)
    rho = torch.as_tensor(np.asarray(c["phantom"]["density"], np.float64)).cuda()
    V = c["phantom"]["dx"] * c["phantom"]["dy"] * c["phantom"]["dz"]
    exp = torch.where(rho > 0, acc.double() / 2.0 ** 32 / (torch.clamp(rho, min=1e-30) * V * 2_100_000), torch.zeros_like(rho))
    assert torch.allclose(dose, exp, rtol=1e-14, atol=0)
    d = acc.cpu().numpy().reshape(120, 256, 256)
    assert d[50:70, 118:138, 118:138].mean() > 5 * d[50:70, :20, :20].mean()


def test_history_ids_beyond_32_bits(B, orc, gpsl, opsl, cfg):
    """A slice of a 2^33-history run: history ids, the Philox counter words and the group offsets are 64-bit on both sides."""
    import torch
    c = cfg("C0")
    N = 1 << 33
    dph, oph = B.DevicePhantom(c["phantom"]), orc.Phantom(c["phantom"])
    assert np.array_equal(gpsl("C0").allocate(N), opsl("C0").allocate(N))
    for hb in (N - 20_000, (1 << 32) - 10_000):
        he = hb + 20_000
        fp = torch.zeros(he - hb, dtype=torch.int64, device="cuda")
        acc = torch.zeros(dph.nvox, dtype=torch.int64, device="cuda")
        gpsl("C0").dose(dph, c["beams"][0], N, 77, batch=6000, dose_acc=acc, fingerprints=fp, history_begin=hb, history_end=he)
        oacc = np.zeros(oph.nvox, np.int64)
        _, _, ofp = opsl("C0").dose(oph, c["beams"][0], N, 77, h_begin=hb, h_end=he, acc=oacc, fingerprints=True)
        assert (fp.cpu().numpy().view(np.uint64) == ofp).mean() >= 0.999
        a = acc.cpu().numpy()
        assert abs(int(a.sum()) - int(oacc.sum())) <= 2e-3 * int(oacc.sum())
    got = gpsl("C0").sample_debug(c["beams"][0], N, 77, (1 << 32) - 5, 10).cpu().numpy().astype(np.float64)
    ref = opsl("C0").sample(c["beams"][0], N, 77, (1 << 32) - 5, 10)
    assert np.allclose(got[0, :, :3], ref[:, :3], atol=2e-5) and np.array_equal(got[1, :, 3], ref[:, 7])


def test_full_size_c1_in_the_bench_configuration(B, orc, gpsl, opsl, cfg):
    """BASELINE.json configs[1] at its full 1e7 histories in the launch configuration bench.py times (the default batch and
    pipelines, sorted order): (a) the interaction sequences of sampled history ranges match the oracle history by
    history; (b) the dose grid is bit-identical to a serial small-batch run; (c) the ledger identities hold."""
    import torch
    c = cfg("C1")
    N, seed = c["n_histories"], c["seed"]
    assert N == 10_000_000
    dph, oph = B.DevicePhantom(c["phantom"]), orc.Phantom(c["phantom"])
    fp = torch.zeros(N, dtype=torch.int64, device="cuda")
    acc = torch.zeros(dph.nvox, dtype=torch.int64, device="cuda")
    gpsl("C1").dose(dph, c["beams"][0], N, seed, batch=B.DEFAULT_BATCH, dose_acc=acc, fingerprints=fp)
    st = B.stats()
    L = st["ledger"]
    assert int(acc.sum().item()) == L["deposited"]
    assert abs(L["deposited"] + L["escaped"] + L["jaw"] - L["incident"]) <= 1e-5 * L["incident"]
    # (a) 64 equally spaced ranges of 2000 histories: all three sub-sources, all energy bins
    gfp = fp.cpu().numpy().view(np.uint64)
    same = total = 0
    oacc = np.zeros(oph.nvox, np.int64)
    for i in range(64):
        a = int(i * N / 64) + 137
        _, _, ofp = opsl("C1").dose(oph, c["beams"][0], N, seed, h_begin=a, h_end=a + 2000, acc=oacc, fingerprints=True)
        same += int((gfp[a:a + 2000] == ofp).sum()); total += 2000
    last = N - 1500                                                        # the contamination-electron tail
    _, _, ofp = opsl("C1").dose(oph, c["beams"][0], N, seed, h_begin=last, h_end=N, acc=oacc, fingerprints=True)
    same += int((gfp[last:] == ofp).sum()); total += N - last
    assert same / total >= 0.999, same / total
    # (b) same bits without fingerprints (the plain kernel variants bench.py times), and serial with a small batch
    acc2 = torch.zeros_like(acc)
    gpsl("C1").dose(dph, c["beams"][0], N, seed, batch=B.DEFAULT_BATCH, dose_acc=acc2)
    assert torch.equal(acc, acc2)
    acc3 = torch.zeros_like(acc)
    gpsl("C1").dose(dph, c["beams"][0], N, seed, batch=1 << 18, dose_acc=acc3, pipelines=1)
    assert torch.equal(acc, acc3) and B.stats()["ledger"] == L


def test_ledgers_beyond_64_bits(B, gpsl, cfg):
    """2^33 histories on C0: the energy ledgers pass 2^64 quanta (128-bit sums in the control block, folded on the host);
    the integer identity sum(acc) == deposited and energy conservation still hold, and the result is the sum of two halves."""
    import torch
    c = cfg("C0")
    dph = B.DevicePhantom(c["phantom"])
    N = 1 << 33
    acc = torch.zeros(dph.nvox, dtype=torch.int64, device="cuda")
    gpsl("C0").dose(dph, c["beams"][0], N, 3, batch=1 << 23, dose_acc=acc)
    L = B.stats()["ledger"]
    assert L["incident"] > 1 << 64 and L["deposited"] > 1 << 62
    total = sum(int(v) for v in acc.cpu().numpy().astype(object))
    assert total == L["deposited"]
    assert abs(L["deposited"] + L["escaped"] + L["jaw"] - L["incident"]) <= 1e-5 * L["incident"]
    acc2 = torch.zeros_like(acc)
    led = 0
    for hb, he in ((0, N // 2), (N // 2, N)):
        gpsl("C0").dose(dph, c["beams"][0], N, 3, batch=B.DEFAULT_BATCH, dose_acc=acc2, history_begin=hb, history_end=he)
        led += B.stats()["ledger"]["deposited"]
    assert torch.equal(acc, acc2) and led == L["deposited"]


# ---------------------------------------------------------------- degenerate inputs
def test_degenerate_phantoms_and_sources(B, orc, cfg, wl):
    """All-vacuum and single-voxel phantoms, an off-axis asymmetric field, and a model whose electron sub-source has no
    weight: tables bit-exact, sequences and ledgers as the oracle's."""
    c = cfg("C1", False)
    # (1) off-axis asymmetric jaws
    jaws = dict(c["jaws"], x1=1.0, x2=6.0, y1=-3.0, y2=0.5)
    g, o = B.Psl(c["psr"], jaws, 16), orc.Psl(c["psr"], jaws, 16)
    ex = g.export()
    assert np.array_equal(ex["rect"], o.rect())
    for gi, gg in enumerate(ex["groups"]):
        og = o.group(gi)
        assert gg["W"] == og["W"] and all(np.array_equal(gg[k], og[k]) for k in ("ring", "sector", "thresh", "alias"))
    n = 40
    ph = dict(nx=n, ny=n, nz=n, dx=0.5, dy=0.5, dz=0.5, ox=-10.0, oy=-10.0, oz=0.0,
              density=np.ones(n ** 3, np.float32), material=np.zeros(n ** 3, np.uint8))
    same, _, _ = compare_with_oracle(B, orc, g, o, ph, c["beams"][0], 300_000, 5, batch=1 << 16, frac_vox=0.98)
    acc = gpu_dose(B, g, B.DevicePhantom(ph), c["beams"][0], 300_000, 5, 1 << 16, want_fp=False)[0].reshape(n, n, n)
    assert acc[:, :, 22:32].sum() > 20 * acc[:, :, 0:10].sum()               # the dose sits at positive x
    # (2) all vacuum: nothing is deposited, everything that passes the jaws escapes
    vac = dict(ph, density=np.zeros(n ** 3, np.float32))
    dph = B.DevicePhantom(vac)
    acc, dose, st, fp = gpu_dose(B, g, dph, c["beams"][0], 50_000, 6, 1 << 14)
    oacc, ores, ofp = o.dose(orc.Phantom(vac), c["beams"][0], 50_000, 6, fingerprints=True)
    # (primaries sampled below the 50 keV cut-off are absorbed in their entry voxel even in vacuum: energy deposited, dose 0)
    assert not dose.any() and np.array_equal(fp, ofp) and np.array_equal(acc != 0, oacc != 0)
    assert abs(st["ledger"]["deposited"] - ores["ledger"]["deposited"]) <= 1e-6 * ores["ledger"]["incident"]
    assert st["ledger"]["deposited"] < 1e-3 * st["ledger"]["incident"] and st["n_flights"] == 0
    assert st["ledger"]["deposited"] + st["ledger"]["escaped"] + st["ledger"]["jaw"] == st["ledger"]["incident"]
    # (3) one voxel
    one = dict(nx=1, ny=1, nz=1, dx=30.0, dy=30.0, dz=30.0, ox=-15.0, oy=-15.0, oz=0.0,
               density=np.ones(1, np.float32), material=np.zeros(1, np.uint8))
    acc, dose, st, fp = gpu_dose(B, g, B.DevicePhantom(one), c["beams"][0], 50_000, 7, 1 << 14)
    oacc, ores, ofp = o.dose(orc.Phantom(one), c["beams"][0], 50_000, 7, fingerprints=True)
    assert (fp == ofp).mean() >= 0.999 and abs(int(acc[0]) - int(oacc[0])) <= 1e-3 * int(oacc[0]) and int(acc[0]) == st["ledger"]["deposited"]
    # (4) a sub-source without weight: its groups are empty, its histories do not exist
    psr = dict(c["psr"], W=np.array(c["psr"]["W"], copy=True))
    psr["W"][2] = 0.0
    g2, o2 = B.Psl(psr, c["jaws"], 16), orc.Psl(psr, c["jaws"], 16)
    N = 100_000
    off = g2.allocate(N)
    assert np.array_equal(off, o2.allocate(N)) and off[2 * psr["n_ebin"]] == N
    acc, dose, st, fp = gpu_dose(B, g2, B.DevicePhantom(ph), c["beams"][0], N, 8, 1 << 15)
    oacc, ores, ofp = o2.dose(orc.Phantom(ph), c["beams"][0], N, 8, fingerprints=True)
    assert st["n_hist"] == ores["n_hist"] and st["n_hist"][2] == 0 and (fp == ofp).mean() >= 0.999


@pytest.mark.parametrize("name,beam,seed", [("C2", 0, 3), ("C3", 3, 43), ("C4", 0, 5)])
def test_full_size_sampled_parity_c2_c3_c4(name, beam, seed, B, orc, cfg):
    """BASELINE.json's other configurations at their full history counts (1e8, 1e8 per beam, 1e9) in the bench launch
    configuration: the fingerprints of sampled history ranges against the oracle, and the ledger identities."""
    import torch
    c = cfg(name)
    N = c["n_histories"]
    g, o = B.Psl(c["psr"], c["jaws"], c["n_sectors"]), orc.Psl(c["psr"], c["jaws"], c["n_sectors"])
    dph, oph = B.DevicePhantom(c["phantom"]), orc.Phantom(c["phantom"])
    fp = torch.zeros(N, dtype=torch.int64, device="cuda")
    acc = torch.zeros(dph.nvox, dtype=torch.int64, device="cuda")
    g.dose(dph, c["beams"][beam], N, seed, batch=B.DEFAULT_BATCH, dose_acc=acc, fingerprints=fp)
    L = B.stats()["ledger"]
    assert int(acc.sum().item()) == L["deposited"]
    assert abs(L["deposited"] + L["escaped"] + L["jaw"] - L["incident"]) <= 1e-5 * L["incident"]
    same = total = 0
    oacc = np.zeros(oph.nvox, np.int64)
    for i in range(48):
        a = int(i * N / 48) + 911
        gfp = fp[a:a + 1000].cpu().numpy().view(np.uint64)
        _, _, ofp = o.dose(oph, c["beams"][beam], N, seed, h_begin=a, h_end=a + 1000, acc=oacc, fingerprints=True)
        same += int((gfp == ofp).sum()); total += 1000
    _, _, ofp = o.dose(oph, c["beams"][beam], N, seed, h_begin=N - 1000, h_end=N, acc=oacc, fingerprints=True)
    same += int((fp[N - 1000:].cpu().numpy().view(np.uint64) == ofp).sum()); total += 1000
    assert same / total >= 0.999, same / total


def test_hierarchical_phantom_on_odd_grids(B, orc, cfg):
    """The brick / super-brick tables on grids whose sizes are no multiples of 4 or 16 (clipped cells at the edges), uniform
    (read through the tables) and with one foreign voxel per super-brick (mostly mixed super-bricks: read directly), and a slab
    phantom whose faces cut through bricks: sequences, counters, ledgers and dose as the oracle's in all three."""
    c = cfg("C1", False)
    g, o = B.Psl(c["psr"], c["jaws"], 16), orc.Psl(c["psr"], c["jaws"], 16)
    nx, ny, nz = 37, 26, 45
    base = dict(nx=nx, ny=ny, nz=nz, dx=0.4, dy=0.5, dz=0.3, ox=-7.4, oy=-6.5, oz=0.0)
    rho = np.ones((nz, ny, nx), np.float32); mat = np.zeros((nz, ny, nx), np.uint8)
    uniform = dict(base, density=rho.reshape(-1).copy(), material=mat.reshape(-1).copy())
    compare_with_oracle(B, orc, g, o, uniform, c["beams"][0], 200_000, 21, batch=1 << 15, frac_vox=0.98)
    rho2 = rho.copy(); rho2[::16, ::16, ::16] = 1.0001                     # one voxel per super-brick differs: every super-brick mixed
    speck = dict(base, density=rho2.reshape(-1).copy(), material=mat.reshape(-1).copy())
    compare_with_oracle(B, orc, g, o, speck, c["beams"][0], 200_000, 21, batch=1 << 15, frac_vox=0.98)
    rho3 = rho.copy(); mat3 = mat.copy()
    rho3[10:17], mat3[10:17] = 1.85, 2                                     # slab faces inside bricks (10, 17 are no multiples of 4)
    rho3[17:30], mat3[17:30] = 0.26, 1
    slab = dict(base, density=rho3.reshape(-1).copy(), material=mat3.reshape(-1).copy())
    compare_with_oracle(B, orc, g, o, slab, c["beams"][0], 200_000, 22, batch=1 << 15, frac_vox=0.98)
