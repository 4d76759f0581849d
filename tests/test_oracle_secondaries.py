"""Pins for the oracle's secondaries (P5, P6): the Compton recoil electron, the pair-production energy
split and the two annihilation photons.  Each is checked against what physics fixes, not against the oracle's own
formula: free-electron Compton scattering conserves momentum (E d = E' d' + p_e d_e with p_e = sqrt(T (T + 2 m_e)));
pair production conserves energy with a uniform split; annihilation at rest gives two 0.511 MeV photons exactly
back to back, isotropic.  A wrong sign, a swapped operand or a dropped term in any of them fails here.

Read from orc.trace with the birth flag (2): a 'B' event carries the position, direction and energy a track starts with.
"""
import math

import numpy as np
import pytest
from scipy import stats

from test_oracle_physics import one_voxel

ME = 0.51099895
BIRTH = 2


def by_track(events):
    out = {}
    for e in events:
        out.setdefault(e["track"], []).append(e)
    return out


def compton_events(orc, ph, E0, n_hist, seed):
    """Yields (E, d, E', d', T, d_e or None) for every Compton scatter of the primaries' whole family."""
    for h in range(n_hist):
        ev = orc.trace(ph, 0, [0, 0, 0, 0.6, 0.0, 0.8, E0, 0], h, seed, flags=BIRTH, max_events=4000)
        tracks = by_track(ev)
        for tid, evs in tracks.items():
            if evs[0]["code"] != "B" or len(evs) < 2:
                continue
            if not any(e["code"] in "CVPX" for e in evs[1:]):
                continue                                   # an electron track
            d, n_child = evs[0]["dir"], 0
            for i, e in enumerate(evs[1:], start=1):
                if e["code"] == "C":
                    E, dp, ct = e["E"], e["dir"], e["aux"]
                    Ep = evs[i + 1]["E"]                  # the photon's next event carries the scattered energy
                    kid = tracks.get(orc.child_track(tid, n_child, 0))
                    de = kid[0] if kid and kid[0]["code"] == "B" else None
                    yield E, d, Ep, dp, ct, de
                    d, n_child = dp, n_child + 1
                elif e["code"] == "X":
                    n_child += 1


@pytest.mark.parametrize("E0,n_hist", [(0.6, 6000), (2.0, 1500), (6.0, 1200)])
def test_compton_recoil_electron_conserves_momentum(orc, E0, n_hist):
    ph = one_voxel(orc)
    n = n_e = 0
    for E, d, Ep, dp, ct, kid in compton_events(orc, ph, E0, n_hist, 311):
        n += 1
        assert float(np.dot(d, dp)) == pytest.approx(ct, abs=1e-12)                  # the logged angle is the angle turned
        assert 1.0 / Ep - 1.0 / E == pytest.approx((1.0 - ct) / ME, rel=1e-9)          # Compton's relation
        T = E - Ep
        if kid is None:
            assert T < 0.2 + 1e-12                                                     # below the cut-off: deposited on the spot
            continue
        n_e += 1
        assert kid["E"] == pytest.approx(T, rel=1e-12) and T >= 0.2
        pe = math.sqrt(T * (T + 2.0 * ME))
        resid = E * np.asarray(d) - Ep * np.asarray(dp) - pe * np.asarray(kid["dir"])
        assert np.abs(resid).max() < 1e-9 * E, (E, Ep, resid)
        assert float(np.dot(kid["dir"], d)) > 0.0                                      # a recoil electron goes forward
    assert n >= 1000 and n_e >= 300, (n, n_e)


def pair_events(orc, ph, E0, n_hist, seed):
    for h in range(n_hist):
        ev = orc.trace(ph, 0, [0, 0, 0, 0.0, 0.6, 0.8, E0, 0], h, seed, flags=BIRTH, max_events=6000)
        tracks = by_track(ev)
        for tid, evs in tracks.items():
            n_child = 0
            for e in evs:
                if e["code"] == "C":
                    n_child += 1
                elif e["code"] == "X":
                    kids = [tracks.get(orc.child_track(tid, n_child, s)) for s in range(4)]
                    yield e, [k[0] if k else None for k in kids]
                    n_child += 1


def test_pair_split_and_annihilation_photons(orc):
    """E = T- + T+ + 1.022 exactly; T-/(E - 1.022) uniform; two 0.511 MeV photons back to back, isotropic."""
    ph = one_voxel(orc, mat=2, rho=1.85)                     # bone: the largest pair cross-section of the model
    split, cosz, azim = [], [], []
    n = 0
    for e, (em, ep, g1, g2) in pair_events(orc, ph, 6.0, 9000, 97):
        n += 1
        E, Tsum = e["E"], e["E"] - 1.022
        assert g1 is not None and g2 is not None and g1["code"] == "B" and g2["code"] == "B"
        assert g1["E"] == pytest.approx(0.511, abs=1e-15) and g2["E"] == pytest.approx(0.511, abs=1e-15)
        assert np.abs(np.asarray(g1["dir"]) + np.asarray(g2["dir"])).max() < 1e-15              # back to back
        assert np.linalg.norm(g1["dir"]) == pytest.approx(1.0, abs=1e-12)
        assert np.array_equal(g1["pos"], e["pos"]) and np.array_equal(g2["pos"], e["pos"])      # born at the conversion site
        cosz.append(g1["dir"][2]); azim.append(math.atan2(g1["dir"][1], g1["dir"][0]))
        if em is not None and ep is not None:                # both charged tracks above the 200 keV cut-off
            assert em["E"] + ep["E"] + 1.022 == pytest.approx(E, abs=1e-12)
            assert np.allclose(em["dir"], e["dir"], atol=0) and np.allclose(ep["dir"], e["dir"], atol=0)   # both along the photon
            split.append(em["E"] / Tsum)
        elif em is not None:
            assert Tsum - em["E"] < 0.2 + 1e-12              # the positron was deposited locally
        elif ep is not None:
            assert Tsum - ep["E"] < 0.2 + 1e-12
    assert n >= 1000, n
    split = np.asarray(split)
    assert len(split) > 800 and 0.0 < split.min() and split.max() < 1.0 and abs(split.mean() - 0.5) < 0.03
    u = (np.asarray(cosz) + 1.0) / 2.0
    assert stats.kstest(u, "uniform").pvalue > 0.01                                         # cos uniform on [-1, 1]
    assert stats.kstest((np.asarray(azim) + math.pi) / (2 * math.pi), "uniform").pvalue > 0.01
    assert abs(np.mean(cosz)) < 4.0 / math.sqrt(3 * len(cosz))


def test_pair_split_is_uniform_at_fixed_energy(orc):
    """First-generation conversions of 6 MeV photons: T-/(E - 1.022) ~ U(0, 1) (KS on the surviving range)."""
    ph = one_voxel(orc, mat=2, rho=1.85)
    Tsum = 6.0 - 1.022
    lo = 0.2 / Tsum
    fr = []
    for e, (em, ep, g1, g2) in pair_events(orc, ph, 6.0, 9000, 98):
        if abs(e["E"] - 6.0) > 1e-12 or em is None or ep is None:
            continue
        fr.append(em["E"] / Tsum)
    fr = np.asarray(fr)
    assert len(fr) > 500 and fr.min() >= lo and fr.max() <= 1 - lo
    assert stats.kstest((fr - lo) / (1 - 2 * lo), "uniform").pvalue > 0.01
