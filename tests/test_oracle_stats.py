"""Pins of oracle/stats.py (PAPER.md:183-189 statistics) against closed forms and library routines."""
import numpy as np
import scipy.stats

from oracle import stats as S


def test_regular_and_poisson_trains():
    # neuron 0: one spike every 50 steps (200 Hz at 0.1 ms); neuron 1: Poisson with p = 0.02 per step; neuron 2: two spikes
    rng = np.random.default_rng(1)
    t0 = np.arange(7, 100000, 50); t1 = np.nonzero(rng.random(100000) < 0.02)[0]; t2 = np.array([10, 500])
    steps = np.concatenate([t0, t1, t2]); ids = np.concatenate([np.zeros_like(t0), np.ones_like(t1), np.full_like(t2, 2)])
    rate, cv = S.rate_cv(steps, ids, 4, 0, 100000, 0.1)
    assert rate[0] == 200.0 and cv[0] == 0.0                              # regular: CV exactly 0
    assert abs(rate[1] - 200.0) < 10 and abs(cv[1] - np.sqrt(1 - 0.02)) < 0.05      # geometric ISI: CV = sqrt(1 - p)
    assert rate[2] == 0.2 and np.isnan(cv[2]) and rate[3] == 0 and np.isnan(cv[3])
    # library routine on the same intervals
    assert cv[1] == np.float64(scipy.stats.variation(np.diff(t1).astype(float)))
    # window: only spikes in [start, end)
    r2, _ = S.rate_cv(steps, ids, 4, 50000, 100000, 0.1)
    assert r2[0] == 200.0 and r2[2] == 0.0


def test_correlation_special_cases_and_numpy():
    rng = np.random.default_rng(2)
    b = rng.poisson(0.3, size=(6, 4000)).astype(float)
    b[1] = b[0]                                   # identical trains
    b[2] = b[0].max() - b[0]                      # complementary train
    b[5] = 1.0                                    # no variance
    C = S.correlation(b)
    assert np.allclose(np.diag(C)[:5], 1.0) and C[0, 1] == 1.0 and abs(C[0, 2] + 1.0) < 1e-12
    assert np.all(np.isnan(C[5])) and np.all(np.isnan(C[:, 5]))
    assert abs(C[3, 4]) < 0.06                    # independent Poisson trains
    ref = np.corrcoef(b[:5])
    assert np.allclose(C[:5, :5], ref, atol=1e-12) and np.allclose(C[:5, :5], C[:5, :5].T)


def test_binning():
    steps = np.array([0, 19, 20, 39, 40, 45, 1000, 5]); ids = np.array([3, 3, 3, 3, 3, 3, 3, 4])
    b = S.binned_trains(steps, ids, [3, 4, 9], 0, 3, 20)
    assert b.tolist() == [[2, 2, 2], [1, 0, 0], [0, 0, 0]]            # the spike at step 1000 falls outside the bins
    b = S.binned_trains(steps, ids, [3], 20, 2, 20)
    assert b.tolist() == [[2, 2]]
