"""oracle.stats — TEST INFRASTRUCTURE: plain numpy restatement of the three spike-train statistics the paper validates its
simulations with.  Written from the paper's definitions, one neuron / one pair at a time; nothing here
is used by the product (the device computes them in `stat_on_spike` / `stat_rate_cv_kernel` / `stat_corr_kernel`).

  rate    average firing rate of the single neuron = spikes / observation time
  CV ISI  "the ratio between the standard deviation and the average of the inter-spike time intervals" (population
          standard deviation; NaN with fewer than two intervals)
  C[i,j]  = <b_i - mu_i, b_j - mu_j> / sqrt(<b_i - mu_i, b_i - mu_i> <b_j - mu_j, b_j - mu_j>), b = spike train
          re-binned to `bin_steps` time steps, mu = its mean, <,> the scalar product
Pins (tests/test_oracle_stats.py): regular trains (CV = 0, known rate), Poisson trains (CV -> 1, C -> 0), identical and
complementary trains (C = +1 / -1), numpy.corrcoef and scipy.stats.variation on random trains.
"""
from __future__ import annotations

import numpy as np


def rate_cv(steps, ids, n_neurons: int, start_step: int, end_step: int, dt_ms: float):
    """Spikes with start_step <= step < end_step.  Returns (rate_hz[n], cv_isi[n])."""
    steps = np.asarray(steps, np.int64); ids = np.asarray(ids, np.int64)
    T_s = (end_step - start_step) * dt_ms * 1e-3
    rate = np.zeros(n_neurons); cv = np.full(n_neurons, np.nan)
    keep = (steps >= start_step) & (steps < end_step)
    steps, ids = steps[keep], ids[keep]
    order = np.lexsort((steps, ids))
    steps, ids = steps[order], ids[order]
    bounds = np.searchsorted(ids, np.arange(n_neurons + 1))
    for i in range(n_neurons):
        t = steps[bounds[i]:bounds[i + 1]]
        rate[i] = t.size / T_s
        if t.size >= 3:
            isi = np.diff(t).astype(np.float64)
            mean = isi.sum() / isi.size
            std = np.sqrt(((isi - mean) ** 2).sum() / isi.size)
            cv[i] = std / mean
    return rate, cv


def binned_trains(steps, ids, sample_ids, start_step: int, n_bins: int, bin_steps: int) -> np.ndarray:
    steps = np.asarray(steps, np.int64); ids = np.asarray(ids, np.int64)
    b = np.zeros((len(sample_ids), n_bins))
    for r, i in enumerate(sample_ids):
        t = steps[ids == i]
        k = (t - start_step) // bin_steps
        k = k[(t >= start_step) & (k < n_bins)]
        for kk in k.tolist():
            b[r, kk] += 1.0
    return b


def correlation(b: np.ndarray) -> np.ndarray:
    """The paper's C[i,j] written out; NaN where a train has no variance."""
    ns = b.shape[0]
    C = np.full((ns, ns), np.nan)
    d = b - b.mean(axis=1, keepdims=True)
    for i in range(ns):
        for j in range(ns):
            den = np.sqrt(np.dot(d[i], d[i]) * np.dot(d[j], d[j]))
            if den > 0:
                C[i, j] = np.dot(d[i], d[j]) / den
    return C
