"""Pins for the oracle's Woodcock flights, interaction selection and electron condensed history."""
import math

import numpy as np
import pytest
from scipy import integrate, stats

from test_oracle_physics import NE, CPHOTO, PPAIR, kn_total_quad, mu_quad, one_voxel, pencil, slab

ME = 0.51099895
X0 = (36.08, 36.08, 27.2)


# ---------------------------------------------------------------- Woodcock: exp(-mu x)
def test_transmission_homogeneous_slab(orc):
    """north_star check 3: narrow-beam transmission through homogeneous water = exp(-mu x) to 0.2 %."""
    n = 4_000_000
    for E, x in ((1.0, 10.0), (3.0, 15.0)):
        ph = slab(orc, [(x, 1.0, 0)])
        _, res, _ = orc.transport(ph, 0, pencil(n, E), 0, 21, flags=1)
        T = res["n_uncollided_escape"] / n
        ref = math.exp(-mu_quad(0, 1.0, E) * x)
        assert T == pytest.approx(ref, rel=2e-3)
        assert res["n_virtual"] == 0                       # homogeneous: every collision is real


def test_transmission_layered_slab_exercises_virtual_collisions(orc):
    """Same through the C2 layers (water 3, bone 2 at 1.85, lung 7 at 0.26, water 4): exp(-sum mu_i t_i)."""
    layers = [(3.0, 1.0, 0), (2.0, 1.85, 2), (7.0, 0.26, 1), (4.0, 1.0, 0)]
    ph = slab(orc, layers)
    n = 4_000_000
    for E in (0.5, 3.0):
        _, res, _ = orc.transport(ph, 0, pencil(n, E), 0, 22, flags=1)
        tau = sum(mu_quad(m, rho, E) * t for t, rho, m in layers)
        assert res["n_uncollided_escape"] / n == pytest.approx(math.exp(-tau), rel=2e-3)
        assert res["n_virtual"] > 0.2 * res["n_flights"]


def test_interaction_fractions_equal_mu_ratios(orc):
    """First-collision type in water while bone (rho 1.85) sets mu_max: V : C : tau : kappa."""
    big = 4000.0
    ph = dict(nx=2, ny=1, nz=1, dx=big, dy=big, dz=big, ox=-big, oy=-big / 2, oz=-big / 2,
              density=np.array([1.0, 1.85], np.float32), material=np.array([0, 2], np.uint8))
    ph = orc.Phantom(ph)
    E, n = 4.0, 40000
    cw = orc.mu_over_rho(0, E) * 1.0
    mmax = 1.85 * orc.mu_over_rho(2, E).sum()
    expect = np.array([mmax - cw.sum(), cw[0], cw[1], cw[2]]) / mmax
    # independent evaluation of the same ratios
    cw_q = np.array([NE[0] * kn_total_quad(E), CPHOTO[0] / E ** 3, PPAIR[0] * math.log(E / 1.022) ** 2])
    mmax_q = mu_quad(2, 1.85, E)
    assert expect == pytest.approx(np.array([mmax_q - cw_q.sum(), *cw_q]) / mmax_q, rel=1e-9)
    counts = {"V": 0, "C": 0, "P": 0, "X": 0}
    start = [-big / 2, 0, 0, 1, 0, 0, E, 0]          # deep inside the water voxel, heading +x
    for h in range(n):
        ev = orc.trace(ph, 0, start, h, 31, flags=1, max_events=4)
        counts[ev[0]["code"]] += 1
    got = np.array([counts[k] for k in "VCPX"], float)
    assert got.sum() == n
    keep = expect * n > 5
    assert stats.chisquare(got[keep], expect[keep] / expect[keep].sum() * got[keep].sum()).pvalue > 0.01
    assert counts["X"] > 0 and counts["V"] > 0


def test_cutoffs_and_pair_bookkeeping(orc):
    ph = one_voxel(orc)
    # photon below 50 keV is absorbed on the spot
    ev = orc.trace(ph, 0, [0, 0, 0, 0, 0, 1, 0.049, 0], 0, 1)
    assert [e["code"] for e in ev] == ["A"]
    # electron below 200 keV likewise
    ev = orc.trace(ph, 1, [0, 0, 0, 0, 0, 1, 0.19, 0], 0, 1)
    assert [e["code"] for e in ev] == ["A"]
    # find a pair event and check children: two charged tracks sharing E - 1.022, two 0.511 photons back to back
    for h in range(3000):
        ev = orc.trace(ph, 0, [0, 0, 0, 0, 0, 1, 6.0, 0], h, 77, max_events=4000)
        if ev[0]["code"] == "X":
            break
    else:
        pytest.fail("no pair event found")
    kids = {}
    for e in ev[1:]:
        kids.setdefault(e["track"], e)
    ids = {s: orc.child_track(0, 0, s) for s in range(4)}
    g2, g3 = kids[ids[2]], kids[ids[3]]
    # first logged event of an annihilation photon carries its pre-event energy 0.511
    assert g2["E"] == pytest.approx(0.511) and g3["E"] == pytest.approx(0.511)
    acc, res, _ = orc.transport(ph, 0, np.array([[0, 0, 0, 0, 0, 1, 6.0, 0]]), h, 77)
    assert res["n_pair"] >= 1 and res["n_sec_photons"] >= 2
    L = res["ledger"]
    assert L["deposited"] + L["escaped"] == pytest.approx(L["incident"], abs=64)


# ---------------------------------------------------------------- electrons
def csda_range(T0, m=0, rho=1.0, Tend=0.2):
    s = (1.0, 1.0, 0.92)[m]
    return integrate.quad(lambda T: 1.0 / (s * (1.52 + 0.25 / T + 0.078 * T) * rho), Tend, T0)[0]


def electron_path(orc, ph, T0, h, fE):
    ev = orc.trace(ph, 1, [0, 0, 0, 0, 0, 1, T0, 0], h, 5, f_e=fE, max_events=100000)
    steps = [e for e in ev if e["code"] in "STAE"]
    return sum(e["aux"] for e in steps if e["code"] in "ST"), steps[-1]["aux"], len(steps), ev


def test_csda_path_length_converges_to_closed_form(orc):
    ph = one_voxel(orc)
    for T0 in (1.0, 2.0, 6.0):
        R = csda_range(T0)
        lo, last, n, _ = electron_path(orc, ph, T0, 0, 0.002)
        assert lo == pytest.approx(R, rel=2e-3) and last < 0.01 * R      # explicit Euler, O(f_E) error
        # default step fraction 0.12: explicit Euler in log T, a few per cent short/long at most
        lo, last, n, _ = electron_path(orc, ph, T0, 0, 0.0)
        assert lo - 1e-12 <= R * 1.08 and lo + last >= R * 0.92
        assert n == pytest.approx(math.log(T0 / 0.2) / -math.log(1 - 0.12), abs=1.5)
    # textbook-order sanity: ranges to zero energy 0.436 / 0.988 / 3.10 cm at 1 / 2 / 6 MeV
    assert csda_range(1.0, Tend=1e-9) == pytest.approx(0.436, abs=0.01)
    assert csda_range(6.0, Tend=1e-9) == pytest.approx(3.10, abs=0.02)


def test_energy_loss_and_voxel_limited_steps(orc):
    """DESIGN.md P7: a condensed step loses 12 % of its starting energy and is cut into sub-steps at voxel
    faces ('S', nudged 1e-4 cm past the face); the deflection happens at its end ('T')."""
    n = 24
    d = 0.25
    ph = orc.Phantom(dict(nx=n, ny=n, nz=n, dx=d, dy=d, dz=d, ox=-3.0, oy=-3.0, oz=0.0,
                          density=np.full(n ** 3, 1.0, np.float32), material=np.zeros(n ** 3, np.uint8)))
    ev = orc.trace(ph, 1, [0.1, 0.1, 0.05, 0, 0, 1, 6.0, 0], 3, 8)
    st = [e for e in ev if e["code"] in "ST"]
    # first sub-step: straight along z from z=0.05 to the face at 0.25 plus eps (s_E = 0.355 > 0.2)
    assert st[0]["code"] == "S" and st[0]["aux"] == pytest.approx(0.2 + 1e-4, abs=1e-12)
    D = 1.52 + 0.25 / 6.0 + 0.078 * 6.0
    assert st[0]["E"] == pytest.approx(6.0 - D * st[0]["aux"], abs=1e-12)
    assert st[0]["pos"][2] == pytest.approx(0.25 + 1e-4, abs=1e-12)
    assert st[0]["dir"] == pytest.approx([0, 0, 1], abs=0)                       # no deflection inside a condensed step
    # second sub-step finishes the 12 % budget with the stopping power at the current energy
    D1 = 1.52 + 0.25 / st[0]["E"] + 0.078 * st[0]["E"]
    assert st[1]["code"] == "T" and st[1]["E"] == pytest.approx(6.0 * 0.88, abs=1e-12)
    assert st[1]["aux"] == pytest.approx((0.72 - D * st[0]["aux"]) / D1, abs=1e-12)
    assert abs(st[1]["dir"][2]) < 1.0
    turns = [e["E"] for e in st if e["code"] == "T"]
    assert len(turns) > 10
    assert np.array(turns[1:]) / np.array(turns[:-1]) == pytest.approx(0.88, abs=1e-12)
    for a, b in zip(st[:-1], st[1:]):
        Dk = 1.52 + 0.25 / a["E"] + 0.078 * a["E"]
        assert a["E"] - b["E"] == pytest.approx(Dk * b["aux"], abs=1e-12)
        assert np.linalg.norm(b["pos"] - a["pos"]) == pytest.approx(b["aux"], abs=1e-12)
        assert b["pos"] - a["pos"] == pytest.approx(b["aux"] * a["dir"], abs=1e-12)      # moves along the pre-step direction
        if b["code"] == "S":
            assert np.array_equal(a["dir"], b["dir"])                                  # sub-steps inside a condensed step do not deflect


def test_multiple_scattering_accumulates_over_the_condensed_step(orc):
    """theta0 uses rho*s/X0 summed over the sub-steps of the condensed step, in every material crossed."""
    from test_oracle_physics import slab
    ph = slab(orc, [(0.25, 1.0, 0), (0.25, 0.26, 1), (3.0, 1.85, 2)])
    T0 = 6.0
    ths = []
    for h in range(4000):
        ev = orc.trace(ph, 1, [0, 0, 0.1, 0, 0, 1, T0, 0], h, 3, max_events=8)
        subs = []
        for e in ev:
            subs.append(e)
            if e["code"] == "T":
                break
        assert [e["code"] for e in subs] == ["S", "S", "T"]
        t = subs[0]["aux"] * 1.0 / 36.08 + subs[1]["aux"] * 0.26 / 36.08 + subs[2]["aux"] * 1.85 / 27.2
        d = subs[-1]["dir"]
        ths.append(math.atan2(math.hypot(d[0], d[1]), d[2]) ** 2 / t)
    pbeta = T0 * (T0 + 2 * ME) / (T0 + ME)
    assert np.mean(ths) == pytest.approx(2 * (13.6 / pbeta) ** 2, rel=5 / math.sqrt(4000))


def test_multiple_scattering_moments(orc):
    """One step: theta = theta0 sqrt(-2 ln U) → <theta^2> = 2 theta0^2 (Highland, no log term), phi uniform."""
    ph = one_voxel(orc)
    T0 = 6.0
    D = 1.52 + 0.25 / T0 + 0.078 * T0
    s = 0.12 * T0 / D
    pbeta = T0 * (T0 + 2 * ME) / (T0 + ME)
    th0 = 13.6 / pbeta * math.sqrt(1.0 * s / X0[0])
    n = 20000
    th, phi = np.empty(n), np.empty(n)
    for h in range(n):
        ev = orc.trace(ph, 1, [0, 0, 0, 0, 0, 1, T0, 0], h, 12, max_events=2)
        assert ev[0]["code"] == "T" and ev[0]["aux"] == pytest.approx(s)
        d = ev[0]["dir"]
        th[h] = math.atan2(math.hypot(d[0], d[1]), d[2])
        phi[h] = math.atan2(d[1], d[0]) % (2 * math.pi)
    assert (th ** 2).mean() == pytest.approx(2 * th0 ** 2, rel=5 * math.sqrt(1.0 / n))
    assert stats.kstest(th ** 2 / (2 * th0 ** 2), "expon").pvalue > 0.01
    assert stats.kstest(phi / (2 * math.pi), "uniform").pvalue > 0.01
