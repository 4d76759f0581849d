"""The gamma-index helper used by the independent-seed GPU test, checked on cases with a known answer."""
import numpy as np

from gamma import gamma_pass_rate


def test_gamma_known_cases():
    z, y, x = np.mgrid[0:20, 0:20, 0:20]
    ref = np.exp(-((x - 10) ** 2 + (y - 10) ** 2) / 30.0) * (1 - z / 40)
    vox = (0.5, 0.5, 0.5)
    assert gamma_pass_rate(ref, ref, vox)[0] == 1.0
    assert gamma_pass_rate(ref, ref * 1.005, vox)[0] == 1.0              # 0.5 % everywhere: inside 1 % of Dmax
    rate, gam = gamma_pass_rate(ref, ref * 1.05, vox)                     # 5 % scale error: fails where the dose is high
    assert rate < 0.9 and gam.max() > 3.0
    assert gamma_pass_rate(ref, np.roll(ref, 1, axis=2), vox)[0] < 0.3    # a 5 mm shift is far outside 1 mm DTA
    # a 1 mm shift along x of a field that is linear in x passes through the distance criterion alone
    lin = 1.0 + 0.02 * x.astype(float)
    shifted = 1.0 + 0.02 * (x - 0.2)                                      # 0.2 voxel = 1 mm
    rate, gam = gamma_pass_rate(lin, shifted, vox, dose_frac=1e-6)
    assert rate > 0.9 and np.median(gam) <= 1.0 + 1e-6
