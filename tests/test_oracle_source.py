"""Pins for the oracle's psl_build, allocation and source sampling (§2.1.1-2.1.3)."""
import math

import numpy as np
import pytest
from scipy import integrate, stats

# Active lets per energy bin, primary / scatter+electron, computed independently in SURVEY.md §8
# (table at the top of §8) with the bounding-box rule — scratch arithmetic of the survey, not this code.
SURVEY_ACTIVE = {"C0": (16, 28), "C1": (144, 240), "C2": (72, 124), "C4": (1976, 2048)}


# ---------------------------------------------------------------- input generator vs quadrature
def test_workload_spectra_and_fluence_match_quadrature(wl):
    phi = [lambda E: E * math.exp(-E / 0.9) * (1 - E / 6), lambda E: E * math.exp(-E / 0.5) * (1 - E / 6),
           lambda E: math.exp(-E / 1.5) * (1 - E / 6)]
    for s in range(3):
        w = wl.spectrum_bins(s, 24)
        tot = integrate.quad(phi[s], 0, 6)[0]
        for e in (0, 3, 11, 23):
            ref = integrate.quad(phi[s], e * 0.25, (e + 1) * 0.25)[0] / tot
            assert w[e] == pytest.approx(ref, rel=1e-9)
    f = lambda r: (1 + 0.04 * r * r) if r <= 12 else (1 + 0.04 * 144) * (16 - r) / 4
    F = wl.fluence_rings(32)
    tot = integrate.quad(lambda r: f(r) * r, 0, 16, points=[12])[0]
    for i in (0, 7, 23, 24, 31):
        ref = integrate.quad(lambda r: f(r) * r, i * 0.5, (i + 1) * 0.5)[0] / tot
        assert F[i] == pytest.approx(ref, rel=1e-9)
    m = wl.psr_model(24, 32)
    assert m["W"].sum() == pytest.approx(1.0, abs=1e-12)
    assert m["W"].sum(axis=(1, 2)) == pytest.approx(wl.SUBSOURCE_WEIGHT, abs=1e-12)


# ---------------------------------------------------------------- psl_build
@pytest.mark.parametrize("name", ["C0", "C1", "C2", "C4"])
def test_active_let_counts_match_survey(name, opsl, cfg):
    psl, c = opsl(name), cfg(name, False)
    ne = c["psr"]["n_ebin"]
    for e in (0, ne - 1):
        assert len(psl.group(0 * ne + e)["ring"]) == SURVEY_ACTIVE[name][0]
        assert len(psl.group(1 * ne + e)["ring"]) == SURVEY_ACTIVE[name][1]
        assert len(psl.group(2 * ne + e)["ring"]) == SURVEY_ACTIVE[name][1]


def test_sampling_rectangles_by_hand(opsl):
    # C1: 10x10 field.  Primary: 5 * 70/100.  Scatter: x edge at the X jaw (z=82): 5*0.82 = 4.1,
    # back-projected from the iso-plane centre: 4.1 * (100-70)/(100-82); y: 3.8 * 30/24.
    r = opsl("C1").rect()
    assert r[0] == pytest.approx([-3.5, 3.5, -3.5, 3.5])
    assert r[1] == pytest.approx([-4.1 * 30 / 18, 4.1 * 30 / 18, -3.8 * 30 / 24, 3.8 * 30 / 24])
    assert r[2] == pytest.approx(r[1])


def test_active_set_toy_by_hand(orc):
    # 2 rings x 4 sectors, ring width 1 cm, off-centre field x in [0.5,1.5], y in [0.2,0.8] on the
    # iso plane with z_phsp = sad (scale 1): only the first-quadrant sector of each ring touches it.
    W = np.ones((3, 1, 2))
    psr = dict(n_ebin=1, n_ring=2, e_min=0.0, e_bin_width=1.0, ring_width=1.0, z_phsp=50.0, W=W,
               sigma_src=(0.1, 1.0, 1.0), z_src=(0.0, 5.0, 5.0), particle_type=(0, 0, 1))
    jaws = dict(x1=1.0, x2=3.0, y1=0.4, y2=1.6, z_jx=60.0, z_jy=55.0, sad=100.0)
    psl = orc.Psl(psr, jaws, 4)
    g = psl.group(0)
    assert psl.rect()[0] == pytest.approx([0.5, 1.5, 0.2, 0.8])
    assert list(zip(g["ring"].tolist(), g["sector"].tolist())) == [(0, 0), (1, 0)]
    # a field on the negative x axis touches sectors 1 and 2 (they share the axis theta = pi)
    jaws2 = dict(x1=-3.0, x2=-2.2, y1=-0.2, y2=0.2, z_jx=60.0, z_jy=55.0, sad=100.0)
    g = orc.Psl(psr, jaws2, 4).group(0)
    assert list(zip(g["ring"].tolist(), g["sector"].tolist())) == [(1, 1), (1, 2)]


def test_active_set_brute_force(opsl, cfg):
    """Every point of the sampling rectangle lies in an active let (the active set is a superset)."""
    rng = np.random.default_rng(5)
    for name in ("C0", "C1", "C2"):
        psl, c = opsl(name), cfg(name, False)
        ne, ns, dr = c["psr"]["n_ebin"], c["n_sectors"], c["psr"]["ring_width"]
        rect = psl.rect()
        for s in range(3):
            g = psl.group(s * ne)
            active = set(zip(g["ring"].tolist(), g["sector"].tolist()))
            x = rng.uniform(rect[s, 0], rect[s, 1], 20000)
            y = rng.uniform(rect[s, 2], rect[s, 3], 20000)
            ring = np.floor(np.hypot(x, y) / dr).astype(int)
            sector = np.floor((np.arctan2(y, x) % (2 * np.pi)) / (2 * np.pi / ns)).astype(int) % ns
            assert set(zip(ring.tolist(), sector.tolist())) <= active
            # and no active let is far from the rectangle: its centre is within one let diagonal
            for (i, k) in active:
                rc, tc = (i + 0.5) * dr, (k + 0.5) * 2 * np.pi / ns
                cx, cy = rc * np.cos(tc), rc * np.sin(tc)
                ddx = max(rect[s, 0] - cx, 0, cx - rect[s, 1])
                ddy = max(rect[s, 2] - cy, 0, cy - rect[s, 3])
                assert math.hypot(ddx, ddy) <= dr + (i + 1) * dr * 2 * np.pi / ns


def test_let_weights_and_alias_reconstruction(opsl, cfg):
    for name in ("C0", "C1", "C4"):
        psl, c = opsl(name), cfg(name, False)
        W, ns, ne = c["psr"]["W"], c["n_sectors"], c["psr"]["n_ebin"]
        for gi in (0, ne + 1, 2 * ne + ne - 1):
            g = psl.group(gi)
            n = len(g["ring"])
            w = W[g["stype"], g["ebin"], g["ring"]] / ns          # Eq. 1-2 integrated over a sector
            assert g["W"] == pytest.approx(w.sum(), rel=1e-12)
            # exact reconstruction of p_i from (thresh, alias)
            t = g["thresh"].astype(np.float64)
            t = np.where(g["thresh"] == 0xFFFFFFFF, 2.0 ** 32, t)
            mass = t.copy()
            np.add.at(mass, g["alias"], 2.0 ** 32 - t)
            p = mass / (n * 2.0 ** 32)
            assert np.abs(p - w / w.sum()).max() < 2.0 ** -31
            assert np.all(g["alias"] < n)
    # all sectors of a ring present → their weights add up to the ring weight
    psl, c = opsl("C4"), cfg("C4", False)
    g = psl.group(c["psr"]["n_ebin"])        # scatter sub-source, every let active
    assert len(g["ring"]) == 64 * 32
    assert g["W"] == pytest.approx(c["psr"]["W"][1, 0].sum(), rel=1e-12)


def test_allocation_eq3(opsl):
    psl = opsl("C1")
    Wg = np.array([psl.group(g)["W"] for g in range(psl.n_groups)])
    for N in (1, 7, 1000, 100_003, 10_000_000):
        off = psl.allocate(N).astype(np.int64)
        n = np.diff(off)
        assert off[0] == 0 and off[-1] == N and np.all(n >= 0)
        assert np.abs(n - N * Wg / Wg.sum()).max() < 1.0
    # tie → lower index: two equal groups, odd N
    n = np.diff(psl.allocate(3).astype(np.int64))
    assert n.sum() == 3


# ---------------------------------------------------------------- sampling
def _beam_frame(c, s):
    b = c["beams"][0]
    pos = s[:, 0:3] - np.array(b["iso"]) + np.array([0, 0, b["sad"]])
    return pos, s[:, 3:6]


def test_energy_and_ring_histograms_chi2(opsl, cfg):
    """north_star check 1: sampled spectrum and fluence vs the analytic PSR densities."""
    psl, c = opsl("C1"), cfg("C1", False)
    N = 400_000
    s = psl.sample(c["beams"][0], N, 11, 0, N)
    grp = np.where(s[:, 7] < 0, -s[:, 7] - 1, s[:, 7]).astype(int)
    ne, ns, dr, dE = 24, 16, 0.5, 0.25
    W = c["psr"]["W"]
    # group (sub-source, energy-bin) counts: Eq. 3, deterministic to within 1
    Wg = np.array([psl.group(g)["W"] for g in range(psl.n_groups)])
    cnt = np.bincount(grp, minlength=psl.n_groups)
    assert np.abs(cnt - N * Wg / Wg.sum()).max() < 1.0
    # energy uniform inside its bin, and inside the right bin
    ebin = grp % ne
    frac = (s[:, 6] - ebin * dE) / dE
    assert frac.min() > 0 and frac.max() <= 1
    assert stats.kstest(frac, "uniform").pvalue > 0.01
    # spectrum on a grid 4x finer than the bins vs the PSL density (piecewise constant per bin)
    prim = grp < ne
    h, _ = np.histogram(s[prim, 6], bins=96, range=(0, 6))
    expect = np.repeat(Wg[:ne] / Wg[:ne].sum(), 4) / 4 * prim.sum()
    keep = expect > 5
    assert stats.chisquare(h[keep], expect[keep] * h[keep].sum() / expect[keep].sum()).pvalue > 0.01
    # ring histogram of primaries vs W_ring * (active sectors of the ring)/n_s
    pos, _ = _beam_frame(c, s)
    r = np.hypot(pos[:, 0], pos[:, 1])
    g0 = psl.group(0)
    act = np.bincount(g0["ring"], minlength=32)
    ring_w = (W[0].sum(axis=0) * act / ns)
    h = np.bincount(np.floor(r[prim] / dr).astype(int), minlength=32)
    keep = ring_w > 0
    assert np.all(h[~keep] == 0)
    assert stats.chisquare(h[keep], ring_w[keep] / ring_w[keep].sum() * h[keep].sum()).pvalue > 0.01
    # uniform in area inside a ring: (r^2 - r0^2)/(r1^2 - r0^2) ~ U(0,1)
    ring = np.floor(r / dr)
    a = (r * r - (ring * dr) ** 2) / (((ring + 1) * dr) ** 2 - (ring * dr) ** 2)
    assert stats.kstest(a[prim][:100000], "uniform").pvalue > 0.01
    th = (np.arctan2(pos[:, 1], pos[:, 0]) % (2 * np.pi)) / (2 * np.pi / ns)
    assert stats.kstest((th - np.floor(th))[prim][:100000], "uniform").pvalue > 0.01
    assert np.abs(pos[:, 2] - 70.0).max() < 1e-9


def test_eq2_cartesian_fluence(opsl, cfg):
    """Eq. 2: p_PSL(x,y) = p_PSR(r)/(2 pi r).  Bin sampled primaries of C4 on a Cartesian
    grid inside the fully active disc and compare with the ring densities integrated over each cell."""
    psl, c = opsl("C4"), cfg("C4", False)
    off = psl.allocate(10 ** 9).astype(np.int64)
    W = c["psr"]["W"]
    ne = 48
    e = 10                                   # one primary group
    g = psl.group(e)
    n = 600_000
    s = psl.sample(c["beams"][0], 10 ** 9, 3, int(off[e]), n)
    assert np.all(np.where(s[:, 7] < 0, -s[:, 7] - 1, s[:, 7]) == e)
    pos, _ = _beam_frame(c, s)
    edges = np.linspace(-9, 9, 10)           # 2 cm cells, r <= 12.7 < 14: every let there is active
    H, _, _ = np.histogram2d(pos[:, 0], pos[:, 1], bins=[edges, edges])
    dr = 0.25
    dens = W[0, e] / (np.pi * (((np.arange(64) + 1) * dr) ** 2 - (np.arange(64) * dr) ** 2))   # per area
    sub = (np.arange(400) + 0.5) / 400 * 2.0
    expect = np.zeros_like(H)
    for i in range(9):
        for j in range(9):
            X, Y = np.meshgrid(edges[i] + sub, edges[j] + sub, indexing="ij")
            expect[i, j] = dens[np.floor(np.hypot(X, Y) / dr).astype(int)].mean() * 4.0
    expect *= n / g["W"]
    assert H.sum() / n == pytest.approx(expect.sum() / n, abs=4 * math.sqrt(0.25 / n))
    assert stats.chisquare(H.ravel(), expect.ravel() * H.sum() / expect.sum()).pvalue > 0.01


def test_source_backprojection_is_gaussian_and_jaws(opsl, cfg, wl):
    """Eq. 4-5: every ray back-projected to its sub-source plane lands on N(0, sigma_s^2)."""
    psl, c = opsl("C1"), cfg("C1", False)
    N = 10_000_000
    off = psl.allocate(N).astype(np.int64)
    j = c["jaws"]
    for s_idx in range(3):
        first = int(off[s_idx * 24 + 4])
        n = min(60000, int(off[s_idx * 24 + 5]) - first)
        s = psl.sample(c["beams"][0], N, 2, first, n)
        pos, d = _beam_frame(c, s)
        zs, sig = wl.Z_SRC[s_idx], wl.SIGMA_SRC[s_idx]
        t = (pos[:, 2] - zs) / d[:, 2]
        xs, ys = pos[:, 0] - t * d[:, 0], pos[:, 1] - t * d[:, 1]
        assert np.linalg.norm(d, axis=1) == pytest.approx(1.0, abs=1e-12)
        for q in (xs, ys):
            assert abs(q.mean()) < 5 * sig / math.sqrt(n)
            assert q.var() == pytest.approx(sig * sig, rel=5 * math.sqrt(2.0 / n))
            assert stats.kstest(q / sig, "norm").pvalue > 0.01
        assert abs(np.corrcoef(xs, ys)[0, 1]) < 5 / math.sqrt(n)
        # jaw decision recomputed from the ray: inside both openings <=> status >= 0
        xj = xs + (j["z_jx"] - zs) / d[:, 2] * d[:, 0]
        yj = ys + (j["z_jy"] - zs) / d[:, 2] * d[:, 1]
        inside = (np.abs(xj) <= 5 * 0.82) & (np.abs(yj) <= 5 * 0.76)
        clear = (np.abs(np.abs(xj) - 4.1) > 1e-9) & (np.abs(np.abs(yj) - 3.8) > 1e-9)
        assert np.all((s[:, 7] >= 0)[clear] == inside[clear])
        assert 0.05 < inside.mean() < 0.999


def test_point_source_limit_and_beam_rotation(orc, cfg, wl):
    c = cfg("C1", False)
    psr = dict(c["psr"])
    psr["sigma_src"] = (0.0, 0.0, 0.0)
    psl = orc.Psl(psr, c["jaws"], 16)
    s = psl.sample(c["beams"][0], 10000, 9, 0, 10000)
    pos, d = _beam_frame(c, s)
    prim = np.abs(s[:, 7]).astype(int) < 24
    # sigma -> 0: d = p/|p| exactly (Eq. 5 with x_s = y_s = 0)
    ref = pos / np.linalg.norm(pos, axis=1)[:, None]
    assert np.abs(d[prim] - ref[prim]).max() < 1e-14
    # with a point source the jaws cut the iso-plane fluence exactly at the field edge
    iso = pos[prim] * (100.0 / 70.0)
    ok = s[prim, 7] >= 0
    assert np.all(np.abs(iso[ok, 0]) <= 5 + 1e-9) and np.all(np.abs(iso[ok, 1]) <= 5 + 1e-9)
    assert np.all((np.abs(iso[~ok, 0]) >= 5 - 1e-9) | (np.abs(iso[~ok, 1]) >= 5 - 1e-9))
    # gantry rotation = rotate the R = I sample
    b = wl.beam_gantry(51.0)
    R = np.array(b["R"]).reshape(3, 3)
    c1 = cfg("C1", False)
    p1 = orc.Psl(c1["psr"], c1["jaws"], 16)
    a = p1.sample(wl.beam_along_z(100.0), 5000, 4, 0, 5000)
    r = p1.sample(b, 5000, 4, 0, 5000)
    pb = a[:, 0:3] + np.array([0, 0, 100.0]) - np.array([0, 0, 100.0])     # iso (0,0,0), sad 100
    assert np.abs(r[:, 0:3] - (pb - 0) @ R.T).max() < 1e-9
    assert np.abs(r[:, 3:6] - a[:, 3:6] @ R.T).max() < 1e-12
    assert np.array_equal(r[:, 6:8], a[:, 6:8])
    # gantry 0 looks down -y: central axis direction is b_z
    assert R[:, 2] == pytest.approx(np.array(wl.beam_gantry(51.0)["R"]).reshape(3, 3)[:, 2])
    assert np.array(wl.beam_gantry(0.0)["R"]).reshape(3, 3)[:, 2] == pytest.approx([0, -1, 0])
