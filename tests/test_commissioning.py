"""The commissioning utilities: the oracle's per-PSR tally against its own 3-D tally, and the
gradient-projection solver of Eq. 8 against an independent NNLS solver and the optimality conditions."""
import numpy as np
import pytest
from scipy import optimize

from paper_1503_01725_b200 import commissioning as com


def test_measurement_index_layout():
    idx, rows = com.measurement_index(32, 32, 32, 0.5, depths_cm=(1.5, 10.0))
    assert rows == 32 + 2 * (31 + 31)                       # depth dose + two profiles per depth, axis voxel counted once
    assert idx[:, 16, 16].tolist() == list(range(1, 33))    # rows 1..32 run down the central axis
    used = idx[idx > 0]
    assert sorted(used.tolist()) == list(range(1, rows + 1))
    assert idx[3, 16, :].min() > 0 and idx[3, :, 16].min() > 0 and idx[20, 16, :].min() > 0
    assert (idx[5] > 0).sum() == 1


def test_oracle_tally_columns_sum_to_the_dose(orc, opsl, cfg):
    """Every deposit goes to exactly one column, so summing the per-PSR matrix over columns must give the ordinary 3-D
    tally at the measurement voxels — exactly (integers); and each history's deposits land in the column of its own
    (sub-source, energy bin, ring)."""
    c = cfg("C0")
    psr = c["psr"]
    o = opsl("C0")
    ph = orc.Phantom(c["phantom"])
    idx, rows = com.measurement_index(32, 32, 32, 0.5, depths_cm=(1.5, 5.0))
    cols = com.n_columns(psr["n_ebin"], psr["n_ring"])
    N = 200_000
    acc, A, res = orc.dose_com(o, ph, c["beams"][0], N, 7, idx.reshape(-1), rows, cols)
    acc_plain, _, _ = o.dose(ph, c["beams"][0], N, 7)
    assert np.array_equal(acc, acc_plain)                   # the tally does not disturb the run
    flat = idx.reshape(-1)
    sel = np.nonzero(flat)[0]
    assert np.array_equal(A.sum(axis=0)[flat[sel] - 1], acc[sel])
    assert A.sum() > 0
    # column structure: in C0 only rings whose sectors touch the 4x4 field are active; electrons share one column per bin
    ne, nr = psr["n_ebin"], psr["n_ring"]
    used_cols = np.nonzero(A.sum(axis=1))[0]
    photon_cols = used_cols[used_cols < 2 * ne * nr]
    active_rings = {int(r) for g in range(2 * ne) for r in o.group(g)["ring"]}
    assert {int(cc % nr) for cc in photon_cols} <= active_rings
    assert orc.com_column(ne, nr, 0, 1, 3, 5) == (1 * ne + 3) * nr + 5 and orc.com_column(ne, nr, 1, 2, 3, 5) == 2 * ne * nr + 3
    # a single history puts everything in one column
    off = o.allocate(N)
    for h in (1, int(off[ne + 2]) + 5):
        _, A1, r1 = orc.dose_com(o, ph, c["beams"][0], N, 7, np.ones(32 ** 3, np.int32), 1, cols, h_begin=h, h_end=h + 1)
        assert (A1.sum(axis=1) != 0).sum() <= 1


@pytest.mark.parametrize("seed", [0, 1, 2])
def test_gradient_projection_solves_eq8(seed):
    rng = np.random.default_rng(seed)
    m, n = 120, 40
    A = rng.random((m, n)) * (rng.random((1, n)) + 0.1)
    x_true = np.where(rng.random(n) < 0.6, rng.random(n) * 2, 0.0)
    b = A @ x_true + (0.0 if seed == 0 else 0.01 * rng.standard_normal(m))
    x, info = com.solve_gradient_projection(A, b, delta=1e-14, max_iter=200000)
    x_ref, rnorm = optimize.nnls(A, b)
    assert np.all(x >= 0)
    assert info["objective"] <= rnorm ** 2 * (1 + 1e-6) + 1e-12           # as good as Lawson-Hanson
    assert np.linalg.norm(A @ x - A @ x_ref) <= 1e-4 * np.linalg.norm(b)   # same fitted dose
    assert all(f1 <= f0 for f0, f1 in zip(info["history"], info["history"][1:]))    # Armijo: monotone descent
    assert info["kkt"] <= 1e-3 * np.abs(2 * A.T @ b).max()


def test_gradient_projection_edge_cases():
    A = np.array([[1.0, 0.0], [0.0, 1.0]])
    x, info = com.solve_gradient_projection(A, np.array([2.0, -3.0]))      # the unconstrained optimum is infeasible in x2
    assert x == pytest.approx([2.0, 0.0], abs=1e-9) and info["objective"] == pytest.approx(9.0, rel=1e-9)
    x, info = com.solve_gradient_projection(A, np.array([1.0, 1.0]))       # starts at the optimum (x0 = 1)
    assert info["iterations"] == 1 and x == pytest.approx([1.0, 1.0])
