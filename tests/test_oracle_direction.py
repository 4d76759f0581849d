"""Pins for the oracle's Eq. 6 / Eq. 7 direction models: the sampled (alpha, beta)
follow the K = 3 Gaussian mixture (scattered photons) and the zero-mean Gaussian (electrons) in closed form, the
component fractions follow c_k / sum c (the cumulative look-up table with the full sum in the denominator), the local
frame has u along the radius, and survivors of the jaw test cross the jaw planes inside the opening."""
import numpy as np
import pytest
from scipy import stats


@pytest.fixture(scope="module")
def setup(orc, cfg, wl):
    c = cfg("C1", False)
    psr = c["psr"]
    jaws = dict(c["jaws"], x1=-30.0, x2=30.0, y1=-30.0, y2=30.0)
    o = orc.Psl(psr, jaws, c["n_sectors"])
    dm = {s: wl.direction_model(s, psr["n_ebin"], psr["n_ring"]) for s in (1, 2)}
    for s in (1, 2):
        o.set_direction_model(s, dm[s]["c"], dm[s]["mu"], dm[s]["sigma_a"], dm[s]["sigma_b"])
    return c, psr, o, dm


def local_angles(rows):
    x, y = rows[:, 0], rows[:, 1]
    r = np.hypot(x, y)
    ct, st = x / r, y / r
    ul, vl = rows[:, 3] * ct + rows[:, 4] * st, -rows[:, 3] * st + rows[:, 4] * ct      # u radial, v tangential
    return r, np.arctan(ul / rows[:, 5]), np.arctan(vl / rows[:, 5])


@pytest.mark.parametrize("stype", [1, 2])
def test_alpha_beta_follow_eq6_eq7(stype, setup):
    c, psr, o, dm = setup
    ne, nr = psr["n_ebin"], psr["n_ring"]
    N = 40_000_000
    off = o.allocate(N).astype(np.int64)
    for e in (2, 15):
        g = stype * ne + e
        cnt = int(min(off[g + 1] - off[g], 1_500_000))
        rows = o.sample(c["beams"][0], N, 21, int(off[g]), cnt)
        r, alpha, beta = local_angles(rows)
        ring = np.minimum(np.floor(r / psr["ring_width"]).astype(int), nr - 1)
        for i in (3, 14, 26):
            sel = ring == i
            if sel.sum() < 2000:
                continue
            ck = dm[stype]["c"][e, i] / dm[stype]["c"][e, i].sum()
            mu, sa, sb = dm[stype]["mu"][e, i], dm[stype]["sigma_a"][e, i], dm[stype]["sigma_b"][e, i]
            cdf_a = lambda a: sum(w * stats.norm.cdf(a, m, s) for w, m, s in zip(ck, mu, sa))
            cdf_b = lambda b: sum(w * stats.norm.cdf(b, 0.0, s) for w, s in zip(ck, sb))
            assert stats.kstest(alpha[sel], cdf_a).pvalue > 1e-3, (stype, e, i)
            assert stats.kstest(beta[sel], cdf_b).pvalue > 1e-3, (stype, e, i)
            # first two moments of the mixture in closed form
            m1 = float((ck * mu).sum()); v = float((ck * (sa ** 2 + mu ** 2)).sum() - m1 ** 2)
            n = int(sel.sum())
            assert abs(alpha[sel].mean() - m1) < 5 * np.sqrt(v / n)
            assert abs(beta[sel].var() - float((ck * sb ** 2).sum())) < 0.05 * float((ck * sb ** 2).sum())
            # alpha and beta are independent inside a component; for K = 1 (Eq. 7) they are uncorrelated overall
            if stype == 2:
                assert abs(np.corrcoef(alpha[sel], beta[sel])[0, 1]) < 5 / np.sqrt(n)


def test_component_fractions_and_jaw_rejection(orc, cfg, wl):
    """A mixture with well separated means makes the component of every sample identifiable: the fractions must be
    c_k / sum_j c_j.  Then, with real jaws, every surviving ray crosses both jaw planes inside the opening and every
    rejected one misses at least one (independent recomputation from the returned position and direction)."""
    c = cfg("C1", False)
    psr = c["psr"]
    ne, nr = psr["n_ebin"], psr["n_ring"]
    o = orc.Psl(psr, c["jaws"], c["n_sectors"])
    cw = np.broadcast_to(np.array([2.0, 5.0, 3.0]), (ne, nr, 3))
    mu = np.broadcast_to(np.array([-0.6, 0.0, 0.6]), (ne, nr, 3))
    sg = np.full((ne, nr, 3), 0.02)
    o.set_direction_model(1, cw, mu, sg, sg)
    N = 20_000_000
    off = o.allocate(N).astype(np.int64)
    rows = o.sample(c["beams"][0], N, 5, int(off[ne + 4]), 400_000)
    r, alpha, beta = local_angles(rows)
    comp = np.digitize(alpha, [-0.3, 0.3])
    counts = np.bincount(comp, minlength=3)
    assert stats.chisquare(counts, np.array([0.2, 0.5, 0.3]) * len(alpha)).pvalue > 1e-3
    # jaw test (realistic widths again)
    dm = wl.direction_model(1, ne, nr)
    o.set_direction_model(1, dm["c"], dm["mu"], dm["sigma_a"], dm["sigma_b"])
    rows = o.sample(c["beams"][0], N, 6, int(off[ne + 4]), 400_000)
    j = c["jaws"]
    zp = psr["z_phsp"]
    x, y = rows[:, 0], rows[:, 1]                                          # C1: R = identity, iso = (0, 0, 0): x, y are plane coordinates
    xj = x + rows[:, 3] / rows[:, 5] * (j["z_jx"] - zp)
    yj = y + rows[:, 4] / rows[:, 5] * (j["z_jy"] - zp)
    inside = (xj >= j["x1"] * j["z_jx"] / j["sad"]) & (xj <= j["x2"] * j["z_jx"] / j["sad"]) & \
             (yj >= j["y1"] * j["z_jy"] / j["sad"]) & (yj <= j["y2"] * j["z_jy"] / j["sad"])
    passed = rows[:, 7] >= 0
    assert 0.02 < passed.mean() < 0.98
    assert (inside == passed).mean() > 1 - 1e-6
