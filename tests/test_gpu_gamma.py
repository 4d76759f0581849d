"""north_star: "With independent seeds, the gamma pass rate at 1 %/1 mm must be at least 99 %."

Run where the statistics allow it (SURVEY §8d caveat): C0 geometry, 1e9 histories on each side, which
leaves sigma ~ 0.3 % of the local dose per voxel above 10 % of Dmax (measured, printed below).  The oracle side runs
as one single-threaded process per host core over disjoint history ranges whose int64 tallies are summed (exact).
Global criterion (1 % of Dmax), 1 mm DTA on a 0.25 mm search lattice."""
import multiprocessing as mp
import os

import numpy as np
import pytest

from gamma import gamma_pass_rate

pytestmark = pytest.mark.gpu

N = 1_000_000_000
SEED_GPU, SEED_ORACLE, SEED_GPU2 = 101, 202, 303


def _oracle_part(args):
    a, b = args
    import oracle
    from paper_1503_01725_b200 import workloads
    c = workloads.make_config("C0")
    o = oracle.Psl(c["psr"], c["jaws"], c["n_sectors"])
    ph = oracle.Phantom(c["phantom"])
    acc = np.zeros(ph.nvox, np.int64)
    o.dose(ph, c["beams"][0], N, SEED_ORACLE, h_begin=a, h_end=b, acc=acc)
    return acc


def test_gamma_independent_seeds_c0(cfg):
    import torch
    from paper_1503_01725_b200 import binding as B
    c = cfg("C0")
    g = B.Psl(c["psr"], c["jaws"], c["n_sectors"])
    dph = B.DevicePhantom(c["phantom"])

    def gpu(seed):
        acc = torch.zeros(dph.nvox, dtype=torch.int64, device="cuda")
        g.dose(dph, c["beams"][0], N, seed, batch=1 << 22, dose_acc=acc)
        return acc.cpu().numpy().astype(np.float64).reshape(32, 32, 32)

    d_gpu, d_gpu2 = gpu(SEED_GPU), gpu(SEED_GPU2)
    procs = max(1, os.cpu_count() or 1)
    parts = 4 * procs
    ranges = [(N * i // parts, N * (i + 1) // parts) for i in range(parts)]
    with mp.get_context("spawn").Pool(procs) as pool:
        acc = sum(pool.map(_oracle_part, ranges))
    d_orc = acc.astype(np.float64).reshape(32, 32, 32)
    big = d_orc > 0.1 * d_orc.max()
    sigma = float(((d_gpu[big] - d_gpu2[big]) / d_orc[big]).std() / np.sqrt(2))
    rate, gam = gamma_pass_rate(d_orc, d_gpu, (0.5, 0.5, 0.5), dose_frac=0.01, dta_cm=0.1, threshold=0.10)
    rate2, _ = gamma_pass_rate(d_gpu2, d_gpu, (0.5, 0.5, 0.5), dose_frac=0.01, dta_cm=0.1, threshold=0.10)
    mean_ratio = float(d_gpu[big].sum() / d_orc[big].sum())
    print("gamma 1%%/1mm GPU(seed %d) vs oracle(seed %d), %g histories each, %d oracle processes: pass %.4f (max gamma %.2f); "
          "GPU vs GPU(seed %d): %.4f; sigma per voxel %.2e of local dose; integral dose ratio %.6f"
          % (SEED_GPU, SEED_ORACLE, N, procs, rate, gam.max(), SEED_GPU2, rate2, sigma, mean_ratio))
    assert sigma < 4e-3
    assert rate >= 0.99 and rate2 >= 0.99
    assert abs(mean_ratio - 1) < 5e-4                       # no bias between the two implementations beyond statistics
