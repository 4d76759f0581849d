"""Pins for the oracle's scoring, ledgers, fingerprints and whole-chain behaviour."""
import numpy as np
import pytest


@pytest.fixture(scope="module")
def c0run(orc, opsl, cfg):
    c = cfg("C0")
    ph = orc.Phantom(c["phantom"])
    acc, res, fp = opsl("C0").dose(ph, c["beams"][0], 100_000, 1, fingerprints=True)
    return c, ph, acc, res, fp


def test_energy_conservation_c0(c0run):
    """north_star check 4: deposited + escaped + jaw-rejected = incident to 1e-6 relative."""
    _, _, acc, res, _ = c0run
    L = res["ledger"]
    assert abs(L["deposited"] + L["escaped"] + L["jaw"] - L["incident"]) / L["incident"] < 1e-6
    assert int(acc.sum()) == L["deposited"]                       # integers: exact
    assert sum(res["n_hist"]) == 100_000
    assert res["n_electron_tracks"] == res["n_sec_electrons"] + res["n_hist"][2] - \
        (res["n_jaw_rejected"] - _rejected_photons(c0run))


def _rejected_photons(c0run):
    c, _, _, res, fp = c0run
    # jaw-rejected histories have the fingerprint of (track 0, 'J'); count those among electron histories
    import oracle
    off = oracle.Psl(c["psr"], c["jaws"], c["n_sectors"]).allocate(100_000).astype(np.int64)
    first_e = int(off[2 * c["psr"]["n_ebin"]])
    v = 0xcbf29ce484222325
    for b in (0, 0, 0, 0, ord("J")):
        v = ((v ^ b) * 0x100000001b3) & (2 ** 64 - 1)
    rej = fp == np.uint64(v)
    assert int(rej.sum()) == res["n_jaw_rejected"]
    return int(rej[:first_e].sum())


def test_conservation_heterogeneous_and_rotated(orc, cfg, wl):
    c = cfg("C1", False)
    psl = orc.Psl(c["psr"], wl.jaws(5.0), 16)
    # small layered phantom with vacuum and all three materials, gantry beam through it
    n = 24
    rho = np.ones((n, n, n), np.float32)
    mat = np.zeros((n, n, n), np.uint8)
    rho[6:10], mat[6:10] = 1.85, 2
    rho[10:16], mat[10:16] = 0.26, 1
    rho[16:18] = 0.0
    ph = orc.Phantom(dict(nx=n, ny=n, nz=n, dx=0.5, dy=0.5, dz=0.5, ox=-6.0, oy=-6.0, oz=-6.0,
                          density=rho.reshape(-1), material=mat.reshape(-1)))
    for beam in (wl.beam_gantry(0.0), wl.beam_gantry(103.0), wl.beam_along_z(94.0)):
        acc, res, _ = psl.dose(ph, beam, 30_000, 6)
        L = res["ledger"]
        assert abs(L["deposited"] + L["escaped"] + L["jaw"] - L["incident"]) / L["incident"] < 1e-6
        assert int(acc.sum()) == L["deposited"] and L["deposited"] > 0
    # beam along +z reaches the vacuum layer only after matter: nothing is deposited in vacuum voxels
    # (a sub-cut-off particle ENTERING through a vacuum voxel is absorbed there by definition, dose 0)
    assert np.all(acc.reshape(n, n, n)[16:18] == 0)


def test_partition_and_order_invariance(orc, opsl, cfg, c0run):
    """A history's result depends only on (seed, history id): any split of the id range sums to the same bits."""
    c, ph, acc, res, fp = c0run
    psl = opsl("C0")
    parts = [(70_000, 100_000), (0, 1), (1, 33_333), (33_333, 70_000)]
    tot = np.zeros_like(acc)
    led = {k: 0 for k in res["ledger"]}
    fps = np.zeros_like(fp)
    for a, b in parts:
        _, r, f = psl.dose(ph, c["beams"][0], 100_000, 1, h_begin=a, h_end=b, acc=tot, fingerprints=True)
        for k in led:
            led[k] += r["ledger"][k]
        fps[a:b] = f
    assert np.array_equal(tot, acc) and led == res["ledger"] and np.array_equal(fps, fp)
    # a different seed gives a different answer
    acc2, _, _ = psl.dose(ph, c["beams"][0], 100_000, 2, h_end=2000)
    acc1, _, _ = psl.dose(ph, c["beams"][0], 100_000, 1, h_end=2000)
    assert not np.array_equal(acc1, acc2)


def test_electrons_local_flag_keeps_energy(orc, opsl, cfg):
    c = cfg("C0")
    ph = orc.Phantom(c["phantom"])
    _, r0, _ = opsl("C0").dose(ph, c["beams"][0], 100_000, 1, h_end=20_000, flags=0)
    _, r1, _ = opsl("C0").dose(ph, c["beams"][0], 100_000, 1, h_end=20_000, flags=1)
    assert r1["n_sec_electrons"] == 0 and r1["n_electron_steps"] == 0
    assert r1["n_compton"] == r0["n_compton"] and r1["n_flights"] == r0["n_flights"]
    L = r1["ledger"]
    assert abs(L["deposited"] + L["escaped"] + L["jaw"] - L["incident"]) / L["incident"] < 1e-6


def test_depth_dose_shape_c1_like(orc, opsl, cfg, wl):
    """Soft sanity of the whole chain (synthetic physics): build-up then fall-off on the central axis."""
    c = cfg("C1", False)
    ph = orc.Phantom(wl.water_cube(64, 0.25))
    acc, res, _ = opsl("C1").dose(ph, c["beams"][0], 400_000, 2)
    d = orc.finalise(ph, acc, 400_000).reshape(64, 64, 64)
    pdd = d[:, 24:40, 24:40].mean(axis=(1, 2))
    k = int(np.argmax(np.convolve(pdd, np.ones(3) / 3, mode="same")))
    assert 2 <= k <= 12                          # maximum between 0.5 and 3 cm
    assert pdd[0] < 0.8 * pdd.max()              # build-up
    assert 0.5 < pdd[40:44].mean() / pdd.max() < 0.85   # ~10 cm depth
    # dose outside the field is small
    assert d[8:56, :4, :4].mean() < 0.1 * pdd.mean()


def test_finalise_units(orc):
    ph = orc.Phantom(dict(nx=2, ny=1, nz=1, dx=0.5, dy=0.2, dz=0.1, ox=0, oy=0, oz=0,
                          density=np.array([2.0, 0.0], np.float32), material=np.zeros(2, np.uint8)))
    acc = np.array([3 << 32, 5 << 32], np.int64)
    d = orc.finalise(ph, acc, 10)
    assert d[0] == pytest.approx(3.0 / (2.0 * 0.01 * 10)) and d[1] == 0.0


def test_dose_list_and_strict_fingerprints(orc, cfg, opsl):
    """orc_dose_list (the tally of a chosen set of histories) equals orc_dose over the same ids; the strict fingerprint
    (FLAG_FP_VOXELS: also voxels, accepted Kahn trial and branch, sub-step kinds) changes no result, differs from the plain
    one exactly for the histories that deposit or scatter, and tells apart two histories the plain one cannot."""
    c = cfg("C0")
    o, ph = opsl("C0"), orc.Phantom(c["phantom"])
    beam, N, seed = c["beams"][0], 100_000, 1
    a1, r1, f1 = o.dose(ph, beam, N, seed, h_begin=2000, h_end=2600, fingerprints=True)
    ids = np.arange(2000, 2600)
    a2, r2, f2 = orc.dose_list(o, ph, beam, N, seed, ids, fingerprints=True)
    assert np.array_equal(a1, a2) and np.array_equal(f1, f2) and r1 == r2
    # a permuted, thinned list: the same per-history fingerprints, the tally of exactly those histories
    pick = np.random.default_rng(5).permutation(ids)[:200]
    a3, _, f3 = orc.dose_list(o, ph, beam, N, seed, pick, fingerprints=True)
    assert np.array_equal(f3, f1[pick - 2000])
    a4 = np.zeros_like(a3)
    for h in pick:
        o.dose(ph, beam, N, seed, h_begin=int(h), h_end=int(h) + 1, acc=a4)
    assert np.array_equal(a3, a4)
    # strict fingerprints: same tally and counters; equal to the plain ones only for histories without a deposit or scatter
    a5, r5, f5 = o.dose(ph, beam, N, seed, h_begin=2000, h_end=2600, flags=orc.FLAG_FP_VOXELS, fingerprints=True)
    assert np.array_equal(a1, a5) and r1 == r5
    same = f5 == f1
    assert 0.2 < same.mean() < 0.8                              # jaw-rejected / missed / escaped-uncollided histories hash the same
    for h in np.flatnonzero(same)[:20]:
        t = np.zeros_like(a1)
        o.dose(ph, beam, N, seed, h_begin=2000 + int(h), h_end=2001 + int(h), acc=t)
        assert not t.any()                                      # ... and they deposit nothing
    for h in np.flatnonzero(~same)[:20]:
        _, rr, _ = o.dose(ph, beam, N, seed, h_begin=2000 + int(h), h_end=2001 + int(h))
        assert rr["n_deposits"] > 0 or rr["n_compton"] > 0
