"""NEXT-3: the commissioning tally on the GPU (per-PSR dose matrix through the 3-D index array)
against the oracle, and the whole commissioning loop (Eq. 8) on a synthetic 'measurement'."""
import numpy as np
import pytest

from test_gpu_parity import B          # noqa: F401
from paper_1503_01725_b200 import commissioning as com

pytestmark = pytest.mark.gpu


def gpu_matrix(B, psl, dph, beam, N, seed, idx, rows, cols, **opt):
    import torch
    acc = torch.zeros(dph.nvox, dtype=torch.int64, device="cuda")
    A = torch.zeros((cols, rows), dtype=torch.int64, device="cuda")
    d_idx = torch.as_tensor(np.ascontiguousarray(idx.reshape(-1), np.int32)).cuda()
    psl.dose(dph, beam, N, seed, dose_acc=acc, com_index=d_idx, com_dose=A, **opt)
    return acc.cpu().numpy(), A.cpu().numpy()


def test_tally_identity_determinism_and_oracle_parity(B, orc, cfg):
    c = cfg("C0")
    psr = c["psr"]
    g, o = B.Psl(psr, c["jaws"], c["n_sectors"]), orc.Psl(psr, c["jaws"], c["n_sectors"])
    dph, oph = B.DevicePhantom(c["phantom"]), orc.Phantom(c["phantom"])
    idx, rows = com.measurement_index(32, 32, 32, 0.5, depths_cm=(1.5, 5.0, 10.0))
    cols = com.n_columns(psr["n_ebin"], psr["n_ring"])
    N, seed = 400_000, 9
    acc, A = gpu_matrix(B, g, dph, c["beams"][0], N, seed, idx, rows, cols, batch=1 << 16)
    flat = idx.reshape(-1)
    sel = np.nonzero(flat)[0]
    # every deposit in a measurement voxel went to exactly one column: integer identity with the 3-D tally
    assert np.array_equal(A.sum(axis=0)[flat[sel] - 1], acc[sel])
    # same bits for another batch size / one pipeline, and the 3-D tally is the one of a run without the matrix
    acc2, A2 = gpu_matrix(B, g, dph, c["beams"][0], N, seed, idx, rows, cols, batch=30_000, pipelines=1)
    assert np.array_equal(A, A2) and np.array_equal(acc, acc2)
    # the tally's own kernel variant (MODE_COM, above) and the stats/fingerprint variant (MODE_DBG) give the same bits
    acc3, A3 = gpu_matrix(B, g, dph, c["beams"][0], N, seed, idx, rows, cols, batch=1 << 15, flags=B.MC_FLAG_STATS)
    assert np.array_equal(A, A3) and np.array_equal(acc, acc3)
    import torch
    plain = torch.zeros(dph.nvox, dtype=torch.int64, device="cuda")
    g.dose(dph, c["beams"][0], N, seed, batch=1 << 16, dose_acc=plain)
    assert np.array_equal(plain.cpu().numpy(), acc)
    # oracle: same seed, same histories
    oacc, OA, _ = orc.dose_com(o, oph, c["beams"][0], N, seed, flat, rows, cols)
    assert np.array_equal(np.nonzero(OA.sum(axis=1))[0], np.nonzero(A.sum(axis=1))[0])      # the same PSR columns are hit
    col_g, col_o = A.sum(axis=1).astype(np.float64), OA.sum(axis=1).astype(np.float64)
    big = col_o > 0.02 * col_o.max()
    assert np.max(np.abs(col_g[big] / col_o[big] - 1)) < 2e-3                                # per-PSR integral dose
    row_g, row_o = A.sum(axis=0).astype(np.float64), OA.sum(axis=0).astype(np.float64)
    bigr = row_o > 0.1 * row_o.max()
    assert np.median(np.abs(row_g[bigr] / row_o[bigr] - 1)) < 1e-3
    with pytest.raises(B.PslmcError):
        gpu_matrix(B, g, dph, c["beams"][0], N, seed, idx, rows, cols + 1, batch=1 << 16)


def test_commissioning_loop_recovers_a_reweighted_beam(B, cfg):
    """PAPER.md:126-149 on synthetic data: A from two fields (a large and a small one), b = A x_true for a known vector of
    PSR correction factors, Eq. 8 solved by gradient projection: the commissioned dose A x reproduces b."""
    c = cfg("C0")
    psr = c["psr"]
    dph = B.DevicePhantom(c["phantom"])
    idx, rows = com.measurement_index(32, 32, 32, 0.5, depths_cm=(1.5, 5.0, 10.0))
    cols = com.n_columns(psr["n_ebin"], psr["n_ring"])
    mats = []
    for field, seed in ((12.0, 31), (4.0, 32)):
        jaws = dict(c["jaws"], x1=-field / 2, x2=field / 2, y1=-field / 2, y2=field / 2)
        g = B.Psl(psr, jaws, c["n_sectors"])
        N = 20_000_000
        _, A = gpu_matrix(B, g, dph, c["beams"][0], N, seed, idx, rows, cols, batch=B.DEFAULT_BATCH)
        w_active = sum(gr["W"] for gr in g.export()["groups"])
        mats.append(A.T.astype(np.float64) * (w_active / N))                     # rows x cols, dose per particle of the whole plane
    A = np.vstack(mats)
    A /= A.max()
    used = A.sum(axis=0) > 0
    rng = np.random.default_rng(3)
    x_true = np.where(used, 1.0 + 0.3 * rng.standard_normal(cols), 0.0).clip(0.2, 2.0) * used
    b = A @ x_true
    x, info = com.solve_gradient_projection(A[:, used], b, delta=1e-13, max_iter=100000)
    fit = A[:, used] @ x
    print("commissioning: %d measurement points, %d PSR columns in use, %d iterations, relative residual %.2e" %
          (A.shape[0], int(used.sum()), info["iterations"], np.linalg.norm(fit - b) / np.linalg.norm(b)))
    assert np.all(x >= 0)
    assert np.linalg.norm(fit - b) <= 1e-3 * np.linalg.norm(b)
    assert np.linalg.norm(A[:, used] @ np.ones(int(used.sum())) - b) > 30 * np.linalg.norm(fit - b)   # far better than the uncommissioned model


def test_tally_costs_little(B, cfg):
    """The commissioning tally runs in its own kernel variant (no counters, no fingerprints): on the paper's two commissioning
    field sizes (40x40 and 5x5 cm2) the run with the tally stays close to the plain run's time (printed)."""
    import torch
    c = cfg("C4")
    psr = c["psr"]
    dph = B.DevicePhantom(c["phantom"])
    idx, rows = com.measurement_index(c["phantom"]["nx"], c["phantom"]["ny"], c["phantom"]["nz"], c["phantom"]["dz"], depths_cm=(1.5, 10.0, 20.0))
    cols = com.n_columns(psr["n_ebin"], psr["n_ring"])
    d_idx = torch.as_tensor(np.ascontiguousarray(idx.reshape(-1), np.int32)).cuda()
    N = 50_000_000
    for field in (40.0, 5.0):
        jaws = dict(c["jaws"], x1=-field / 2, x2=field / 2, y1=-field / 2, y2=field / 2)
        g = B.Psl(psr, jaws, c["n_sectors"])
        acc = torch.zeros(dph.nvox, dtype=torch.int64, device="cuda")
        A = torch.zeros((cols, rows), dtype=torch.int64, device="cuda")
        ms = {}
        for key, opt in (("plain", {}), ("tally", dict(com_index=d_idx, com_dose=A))):
            best = 1e30
            for _ in range(3):
                acc.zero_()
                g.dose(dph, c["beams"][0], N, 77, batch=B.DEFAULT_BATCH, dose_acc=acc, **opt)
                best = min(best, B.stats()["ms_total"])
            ms[key] = best
        print("commissioning tally, %gx%g cm2 field, %g histories: plain %.1f ms (%.3e histories/s), with the tally %.1f ms (%.3e histories/s)"
              % (field, field, N, ms["plain"], N / ms["plain"] * 1e3, ms["tally"], N / ms["tally"] * 1e3))
        assert ms["tally"] <= 1.25 * ms["plain"]                      # (measured 1.0x-1.1x; a timing bound with room for the box's noise)
