"""NEXT-2: the paper's Eq. 6 / Eq. 7 direction models on the GPU path against the oracle."""
import numpy as np
import pytest

from test_gpu_parity import B, check_samples          # noqa: F401
from test_gpu_dose import compare_with_oracle

pytestmark = pytest.mark.gpu


def with_models(B, orc, wl, c, **kw):
    psr = c["psr"]
    g, o = B.Psl(psr, c["jaws"], **kw), orc.Psl(psr, c["jaws"], **kw)
    for s in (1, 2):
        dm = wl.direction_model(s, psr["n_ebin"], psr["n_ring"])
        g.set_direction_model(s, dm["c"], dm["mu"], dm["sigma_a"], dm["sigma_b"])
        o.set_direction_model(s, dm["c"], dm["mu"], dm["sigma_a"], dm["sigma_b"])
    return g, o


@pytest.mark.parametrize("name,kw", [("C1", dict(n_sectors=16)), ("C0", dict(n_sectors=8)), ("C4", dict(n_sectors=32)),
                                     ("C1", dict(n_sectors=0, let_size=0.5))])
def test_direction_model_samples(name, kw, B, orc, cfg, wl):
    c = cfg(name, False)
    g, o = with_models(B, orc, wl, c, **kw)
    N = 50_000_000
    off = o.allocate(N).astype(np.int64)
    ne = c["psr"]["n_ebin"]
    for first, count in ((int(off[ne]), 60_001), (int(off[ne + ne // 2]) - 1000, 30_000), (int(off[2 * ne]) - 500, 20_000),
                         (int(off[2 * ne + 3]), 20_000), (int(off[ne]) - 3000, 6000)):
        # Cartesian lets: the ring of a position is floor(r / dr), an fp32-vs-fp64 floor decision that flips for ~1e-6 of
        # the samples (the neighbouring ring's parameters then give another direction); sector lets carry their ring
        check_samples(B, g, o, c["beams"][0], N, 13, first, min(count, N - first), allow_fraction=5e-5 if kw["n_sectors"] == 0 else 0.0)


def test_direction_model_dose_parity_and_restore(B, orc, cfg, wl):
    """Whole path with Eq. 6-7 sources: the scattered and electron sub-sources only (history range of those groups)."""
    c = cfg("C1")
    g, o = with_models(B, orc, wl, c, n_sectors=16)
    N = 30_000_000
    off = o.allocate(N).astype(np.int64)
    ne = c["psr"]["n_ebin"]
    import torch
    dph, oph = B.DevicePhantom(c["phantom"]), orc.Phantom(c["phantom"])
    hb, he = int(off[ne]), min(int(off[ne]) + 600_000, N)
    fp = torch.zeros(he - hb, dtype=torch.int64, device="cuda")
    acc = torch.zeros(dph.nvox, dtype=torch.int64, device="cuda")
    g.dose(dph, c["beams"][0], N, 17, batch=1 << 18, dose_acc=acc, fingerprints=fp, history_begin=hb, history_end=he,
           flags=B.MC_FLAG_STATS)
    st = B.stats()
    oacc = np.zeros(oph.nvox, np.int64)
    _, ores, ofp = o.dose(oph, c["beams"][0], N, 17, h_begin=hb, h_end=he, acc=oacc, fingerprints=True)
    same = float((fp.cpu().numpy().view(np.uint64) == ofp).mean())
    assert same >= 0.999, same
    assert abs(st["n_jaw_rejected"] - ores["n_jaw_rejected"]) <= max(2, 1e-4 * (he - hb))
    a = acc.cpu().numpy().astype(np.float64)
    big = oacc > 0.1 * oacc.max()
    assert np.median(np.abs(a[big] - oacc[big]) / oacc[big]) < 1e-3
    # the last electron-source histories too
    hb2 = N - 200_000
    fp2 = torch.zeros(N - hb2, dtype=torch.int64, device="cuda")
    g.dose(dph, c["beams"][0], N, 17, batch=1 << 17, dose_acc=acc, fingerprints=fp2, history_begin=hb2, history_end=N)
    _, _, ofp2 = o.dose(oph, c["beams"][0], N, 17, h_begin=hb2, h_end=N, acc=oacc, fingerprints=True)
    assert float((fp2.cpu().numpy().view(np.uint64) == ofp2).mean()) >= 0.999
    # K = 0 restores the focal model: same samples as a fresh handle
    for s in (1, 2):
        g.set_direction_model(s)
    fresh = B.Psl(c["psr"], c["jaws"], 16)
    s1 = g.sample_debug(c["beams"][0], N, 17, hb, 10_000).cpu().numpy()
    s2 = fresh.sample_debug(c["beams"][0], N, 17, hb, 10_000).cpu().numpy()
    assert np.array_equal(s1, s2)
