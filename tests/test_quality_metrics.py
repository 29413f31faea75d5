"""Eq. (10) and Eq. (11) of the paper (workloads/quality.py) on cases with known answers."""
import numpy as np

import workloads
from workloads import quality


def test_snr_matches_its_definition():
    rng = np.random.default_rng(0)
    t = rng.random((16, 16))
    n = 0.1 * rng.standard_normal(t.shape)
    f = t + n
    want = 10 * np.log10(((f - f.mean()) ** 2).sum() / (n ** 2).sum())
    assert np.isclose(quality.snr_db(f, t), want)
    # halving the error adds 20 log10(2) dB when the image itself hardly changes
    t2 = np.zeros((64, 64)); t2[16:48, 16:48] = 1.0
    e = 1e-3 * rng.standard_normal(t2.shape)
    assert abs(quality.snr_db(t2 + 0.5 * e, t2) - quality.snr_db(t2 + e, t2) - 20 * np.log10(2)) < 1e-3


def test_cnr_and_the_tumour_rois():
    cfg = workloads.Config("q", L=128, N=4)
    ph = workloads.make_inputs(cfg)["phantom"][0]
    for i in range(cfg.N):
        sig, bg = quality.tumour_rois(ph[i])
        assert 8 <= sig.sum() <= 70                       # pixels wholly inside the 8 mm disc
        assert np.allclose(ph[i][sig], 0.02) and np.allclose(ph[i][bg], 0.004) and bg.sum() > 100
    sig, bg = quality.tumour_rois(ph[0])
    rng = np.random.default_rng(1)
    f = ph[0] + 0.002 * rng.standard_normal(ph[0].shape)
    assert abs(quality.cnr(f, sig, bg) - 0.016 / 0.002) < 1.0     # |0.02 - 0.004| / sigma
