"""Pins for the oracle's transport physics (P1-P9; cut-offs PAPER.md:161)."""
import math

import numpy as np
import pytest
from scipy import integrate, stats

ME = 0.51099895
RE2 = 7.940787e-26
NE = (3.343e23, 3.343e23, 3.100e23)
CPHOTO = (2.77e-6, 2.77e-6, 2.2e-5)
PPAIR = (9.6e-4, 9.6e-4, 1.3e-3)


def kn_dsigma_dcos(E, c):
    """Klein–Nishina differential cross-section per electron d(sigma)/d(cos theta) (textbook form)."""
    a = E / ME
    k = 1.0 / (1.0 + a * (1.0 - c))                 # E'/E
    return math.pi * RE2 * k * k * (k + 1.0 / k - (1.0 - c * c))


def kn_total_quad(E):
    return integrate.quad(lambda c: kn_dsigma_dcos(E, c), -1, 1, epsabs=0, epsrel=1e-12)[0]


def mu_quad(m, rho, E):
    """Linear attenuation from the quadrature of KN + the model's photo and pair terms."""
    pair = PPAIR[m] * math.log(E / 1.022) ** 2 if E > 1.022 else 0.0
    return rho * (NE[m] * kn_total_quad(E) + CPHOTO[m] / E ** 3 + pair)


def one_voxel(orc, size=2000.0, rho=1.0, mat=0):
    ph = dict(nx=1, ny=1, nz=1, dx=size, dy=size, dz=size, ox=-size / 2, oy=-size / 2, oz=-size / 2,
              density=np.array([rho], np.float32), material=np.array([mat], np.uint8))
    return orc.Phantom(ph)


def slab(orc, layers, nxy=1, wxy=4000.0):
    """layers: list of (thickness_cm, rho, material); one voxel per layer needs equal thickness, so
    build on a 0.25 cm grid."""
    dz = 0.25
    rho, mat = [], []
    for t, r, m in layers:
        n = int(round(t / dz))
        rho += [r] * n
        mat += [m] * n
    ph = dict(nx=nxy, ny=nxy, nz=len(rho), dx=wxy, dy=wxy, dz=dz, ox=-wxy * nxy / 2, oy=-wxy * nxy / 2, oz=0.0,
              density=np.repeat(np.array(rho, np.float32), nxy * nxy), material=np.repeat(np.array(mat, np.uint8), nxy * nxy))
    return orc.Phantom(ph)


def pencil(n, E, z=-1.0):
    p = np.zeros((n, 8))
    p[:, 2] = z
    p[:, 5] = 1.0
    p[:, 6] = E
    return p


# ---------------------------------------------------------------- cross-sections
def test_sigma_kn_closed_form_vs_quadrature_and_textbook(orc):
    for E in (0.05, 0.1, 0.5, 1.0, 3.0, 6.0):
        assert orc.sigma_kn(E) == pytest.approx(kn_total_quad(E), rel=1e-9)
    # textbook: 0.2112 barn per electron at 1 MeV; Thomson limit 8 pi r_e^2 / 3 as E -> 0
    assert orc.sigma_kn(1.0) == pytest.approx(0.2112e-24, rel=1e-3)
    assert orc.sigma_kn(1e-4) == pytest.approx(8 * math.pi * RE2 / 3, rel=1e-3)
    # water mu/rho at 1 MeV ~ 0.0707 cm^2/g (NIST, incoherent-dominated)
    assert orc.mu_over_rho(0, 1.0).sum() == pytest.approx(0.0707, rel=5e-3)


def test_mu_components(orc):
    for m in range(3):
        for E in (0.08, 1.0, 1.022, 2.5, 6.0):
            c = orc.mu_over_rho(m, E)
            assert c[0] == pytest.approx(NE[m] * kn_total_quad(E), rel=1e-9)
            assert c[1] == pytest.approx(CPHOTO[m] / E ** 3, rel=1e-12)
            pair = PPAIR[m] * math.log(E / 1.022) ** 2 if E > 1.022 else 0.0
            assert c[2] == pytest.approx(pair, rel=1e-12, abs=1e-300)
    assert orc.stopping(0, 1.0) == pytest.approx(1.52 + 0.25 + 0.078)
    assert orc.stopping(2, 2.0) == pytest.approx(0.92 * (1.52 + 0.125 + 0.156))


# ---------------------------------------------------------------- Klein–Nishina by Kahn
@pytest.mark.parametrize("E", [0.1, 1.0, 6.0])
def test_kahn_matches_klein_nishina(orc, E):
    """north_star check 2: angular distribution vs the closed form."""
    n = 300_000
    c, ep = orc.kahn(E, 17, 0, n)
    a = E / ME
    assert np.all(c >= -1 - 1e-12) and np.all(c <= 1 + 1e-12)
    assert np.abs(ep - E / (1 + a * (1 - c))).max() < 1e-12          # Compton kinematics
    edges = np.linspace(-1, 1, 41)
    h, _ = np.histogram(c, bins=edges)
    tot = kn_total_quad(E)
    expect = np.array([integrate.quad(lambda x: kn_dsigma_dcos(E, x), edges[i], edges[i + 1])[0] for i in range(40)]) / tot
    assert stats.chisquare(h, expect * n).pvalue > 0.01
    mean_ratio = integrate.quad(lambda x: kn_dsigma_dcos(E, x) / (1 + a * (1 - x)), -1, 1)[0] / tot
    assert (ep / E).mean() == pytest.approx(mean_ratio, abs=5 * (ep / E).std() / math.sqrt(n))


def test_kahn_one_block_per_trial(orc):
    """DESIGN.md R1: the flight is block 2 (words 0, 1), every Kahn trial takes one block (words 0-2) and the photon
    azimuth is word 3 of the accepted trial's block: trace one Compton and recompute."""
    ph = one_voxel(orc)
    ev = orc.trace(ph, 0, [0, 0, 0, 0, 0, 1, 2.0, 0], 5, 99, flags=1)
    assert ev[0]["code"] == "C"
    a = 2.0 / ME
    b = 3                                  # block 2 was the flight (distance, selector)
    while True:
        u = (orc.philox(99, 5, 0, b) >> 8) / 2.0 ** 24
        r1, r2, r3 = u[:3]
        b += 1
        if r1 <= (2 * a + 1) / (2 * a + 9):
            eta = 1 + 2 * a * r2
            ok = r3 <= 4 * (1 / eta - 1 / eta ** 2)
        else:
            eta = (2 * a + 1) / (1 + 2 * a * r2)
            ct = 1 - (eta - 1) / a
            ok = r3 <= 0.5 * (ct * ct + 1 / eta)
        if ok:
            break
    ct = 1 - (eta - 1) / a
    phi = 2 * math.pi * u[3]
    assert ev[0]["aux"] == pytest.approx(ct, abs=1e-14)
    assert ev[0]["E"] == pytest.approx(2.0, abs=0)          # event logged with the pre-collision energy
    st = math.sqrt(max(0.0, 1 - ct * ct))
    assert ev[0]["dir"] == pytest.approx([st * math.cos(phi), st * math.sin(phi), ct], abs=1e-12)


def test_rotate(orc):
    rng = np.random.default_rng(3)
    for _ in range(200):
        d = rng.normal(size=3)
        d /= np.linalg.norm(d)
        th, phi = rng.uniform(0, math.pi), rng.uniform(0, 2 * math.pi)
        r = orc.rotate(d, math.cos(th), math.sin(th), phi)
        assert np.linalg.norm(r) == pytest.approx(1.0, abs=1e-12)
        assert float(r @ d) == pytest.approx(math.cos(th), abs=1e-12)
    # d = +z: azimuth is the plain spherical angle; d = -z mirrors z
    r = orc.rotate([0, 0, 1], math.cos(0.3), math.sin(0.3), 1.1)
    assert r == pytest.approx([math.sin(0.3) * math.cos(1.1), math.sin(0.3) * math.sin(1.1), math.cos(0.3)])
    r = orc.rotate([0, 0, -1], math.cos(0.3), math.sin(0.3), 1.1)
    assert r[2] == pytest.approx(-math.cos(0.3))
    # azimuth about a tilted axis is uniform: phi and phi+pi give mirror images about d
    d = np.array([0.6, 0.0, 0.8])
    r1, r2 = orc.rotate(d, 0.5, math.sqrt(0.75), 0.7), orc.rotate(d, 0.5, math.sqrt(0.75), 0.7 + math.pi)
    assert (r1 + r2) / 2 == pytest.approx(0.5 * d, abs=1e-12)
