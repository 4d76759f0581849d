"""north_star check 5: a single-history trace of the oracle against a hand computation.

The hand computation below is written from the definitions in DESIGN.md (R1, S3-S5, P2-P5), not from the
oracle's code: Philox4x32-10 in Python integers (itself pinned by the known-answer vectors), the source
draw in `math` floats, the Klein-Nishina total cross-section by numerical quadrature of the differential
cross-section (not the closed form the oracle types), and Kahn's rejection replayed draw by draw.  It covers
history 1 of C0 (seed 1), the first history of that run that passes the jaws: source sample, phantom entry,
first flight, choice of interaction, Compton kinematics and the energy the photon carries on.
"""
import math

import numpy as np
from scipy import integrate

M32 = 0xFFFFFFFF
ME, RE2 = 0.51099895, 7.940787e-26


def philox(seed, h, track, block):
    c = [block, track, h & M32, h >> 32]
    k = [seed & M32, seed >> 32]
    for _ in range(10):
        p0, p1 = 0xD2511F53 * c[0], 0xCD9E8D57 * c[2]
        c = [(p1 >> 32) ^ c[1] ^ k[0], p1 & M32, (p0 >> 32) ^ c[3] ^ k[1], p0 & M32]
        k = [(k[0] + 0x9E3779B9) & M32, (k[1] + 0xBB67AE85) & M32]
    return c


def block(seed, h, track, j):
    return philox(seed, h, track, j)


def u_co(x):
    return (x >> 8) / 2.0 ** 24


def u_oc(x):
    return ((x >> 8) + 1) / 2.0 ** 24


def sigma_kn_quadrature(E):
    """Integral over the sphere of the Klein-Nishina differential cross-section (cm^2 per electron)."""
    a = E / ME

    def dsig(mu):                              # d sigma / d cos(theta), azimuth integrated
        r = 1.0 / (1.0 + a * (1.0 - mu))       # E'/E
        return math.pi * RE2 * r * r * (r + 1.0 / r - (1.0 - mu * mu))
    return integrate.quad(dsig, -1.0, 1.0, epsabs=0, epsrel=1e-13)[0]


def test_hand_trace_of_one_history(orc, opsl, cfg):
    c = cfg("C0")
    psr, jaws, beam, ns = c["psr"], c["jaws"], c["beams"][0], c["n_sectors"]
    N, seed, h = 100_000, 1, 1
    o = opsl("C0")
    assert philox(seed, h, 0, 2) == orc.philox(seed, h, 0, 2).tolist()          # same generator as the pinned one
    off = o.allocate(N)
    g = int(np.searchsorted(off, h, side="right") - 1)
    grp = o.group(g)
    assert grp["stype"] == 0                                                     # a primary photon

    # ---- source draw (S3-S5; Eq. 4-5)
    x = block(seed, h, 0, 0) + block(seed, h, 0, 1)[:2]                          # blocks 0, 1: the source draws
    m = x[0] * len(grp["ring"])
    col, frac = m >> 32, m & M32
    let = col if frac < int(grp["thresh"][col]) else int(grp["alias"][col])
    ring, sector = int(grp["ring"][let]), int(grp["sector"][let])
    r0, r1 = ring * psr["ring_width"], (ring + 1) * psr["ring_width"]
    r = math.sqrt(r0 * r0 + u_co(x[1]) * (r1 * r1 - r0 * r0))
    th = 2.0 * math.pi * (sector + u_co(x[2])) / ns
    p = (r * math.cos(th), r * math.sin(th), psr["z_phsp"])
    E = psr["e_min"] + grp["ebin"] * psr["e_bin_width"] + u_oc(x[3]) * psr["e_bin_width"]
    rho_s = psr["sigma_src"][0] * math.sqrt(-2.0 * math.log(u_oc(x[4])))
    psi = 2.0 * math.pi * u_co(x[5])
    q = (rho_s * math.cos(psi), rho_s * math.sin(psi), psr["z_src"][0])
    d = [p[i] - q[i] for i in range(3)]
    L = math.sqrt(sum(t * t for t in d))
    d = [t / L for t in d]
    # thin jaws: the ray q -> p extended to each jaw plane
    xj = q[0] + (p[0] - q[0]) * (jaws["z_jx"] - q[2]) / (p[2] - q[2])
    yj = q[1] + (p[1] - q[1]) * (jaws["z_jy"] - q[2]) / (p[2] - q[2])
    assert jaws["x1"] * jaws["z_jx"] / jaws["sad"] <= xj <= jaws["x2"] * jaws["z_jx"] / jaws["sad"]
    assert jaws["y1"] * jaws["z_jy"] / jaws["sad"] <= yj <= jaws["y2"] * jaws["z_jy"] / jaws["sad"]
    pos = [p[0] + beam["iso"][0], p[1] + beam["iso"][1], p[2] - beam["sad"] + beam["iso"][2]]   # R = identity in C0
    row = o.sample(beam, N, seed, h, 1)[0]
    assert row[7] == g
    assert np.allclose(row[:3], pos, rtol=0, atol=1e-12) and np.allclose(row[3:6], d, rtol=0, atol=1e-14)
    assert abs(row[6] - E) < 1e-14

    # ---- transport of that photon (P3-P5), water at density 1
    ev = orc.trace(orc.Phantom(c["phantom"]), 0, row, h, seed)
    assert ev[0]["code"] == "C" and ev[0]["track"] == 0
    t_in = (c["phantom"]["oz"] - pos[2]) / d[2] + 1e-4                           # P4: entry through the k = 0 face, + eps
    mu_c = 1.0 * 3.343e23 * sigma_kn_quadrature(E)
    mu_t = 1.0 * 2.77e-6 / E ** 3
    assert E < 1.022                                                             # no pair term at this energy
    mu = mu_c + mu_t                                                             # homogeneous water: mu_max = mu
    flight = block(seed, h, 0, 2)                                                # transport starts at block 2: one block per event
    s = -math.log(u_oc(flight[0])) / mu
    site = [pos[i] + (t_in + s) * d[i] for i in range(3)]
    assert np.allclose(ev[0]["pos"], site, rtol=0, atol=2e-9), (ev[0]["pos"], site)
    assert u_co(flight[1]) * mu < mu_c                                           # Compton was the interaction chosen
    # Kahn's rejection replayed: one block per trial from block 3 on (words 0-2), word 3 of the accepted trial = azimuth
    a, n = E / ME, 3
    while True:
        trial = block(seed, h, 0, n)
        k1, k2, k3 = (u_co(w) for w in trial[:3])
        n += 1
        if k1 <= (2 * a + 1) / (2 * a + 9):
            eta = 1 + 2 * a * k2
            if k3 <= 4 * (1 / eta - 1 / eta ** 2):
                break
        else:
            eta = (2 * a + 1) / (1 + 2 * a * k2)
            ct = 1 - (eta - 1) / a
            if k3 <= 0.5 * (ct * ct + 1 / eta):
                break
    ct = 1 - (eta - 1) / a
    assert abs(ev[0]["aux"] - ct) < 1e-12                                        # the trace records cos(theta) of the scatter
    assert abs(float(np.dot(ev[0]["dir"], d)) - ct) < 1e-12                      # and the photon really turned by it
    assert abs(ev[1]["E"] - E / eta) < 1e-13                                     # Compton energy E' = E / eta
    # the azimuth is word 3 of the accepted trial's block: the scattered direction's azimuth about d is 2 pi U
    phi = 2.0 * math.pi * u_co(trial[3])
    sxy = math.hypot(d[0], d[1])
    e1 = np.array([d[0] * d[2] / sxy, d[1] * d[2] / sxy, -sxy])                  # the frame of DESIGN.md P8
    e2 = np.array([-d[1] / sxy, d[0] / sxy, 0.0])
    st = math.sqrt(1 - ct * ct)
    want = ct * np.array(d) + st * (math.cos(phi) * e1 + math.sin(phi) * e2)
    assert np.allclose(ev[0]["dir"], want, rtol=0, atol=1e-12)
    # the recoil electron is below the 0.2 MeV cut-off here or is transported as track child(0, 0, 0)
    T = E - E / eta
    tracks = {e["track"] for e in ev}
    assert (T < 0.2) == (orc.child_track(0, 0, 0) not in tracks)
