"""On-device spike statistics against oracle/stats.py evaluated on the spike record of the same run:
per-neuron rate and CV ISI, Pearson correlation matrices of the per-population samples (first neurons of each
population, 2 ms bins), for every delivery kernel / step mode that appends spikes in a different place."""
import numpy as np
import pytest

from oracle import stats as S
from paper_2007_14236_b200 import workloads as W

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    from paper_2007_14236_b200 import binding
    return binding


@pytest.mark.parametrize("mode,kernel", [(3, 0), (0, 3), (0, 1), (2, 1), (0, 4), (0, 5), (2, 6)])
def test_statistics_match_the_spike_record(B, mode, kernel):
    wl = W.microcircuit(scale_div=20, n_steps=6000, indegree_div=2)
    N = wl.n_neurons
    g = B.Sim(0.1, wl.ring_slots, wl.seed, record_spikes=True, max_recorded_spikes=1 << 22)
    wl.apply(g)
    g.set_option(B.OPT_DELIVERY_KERNEL, kernel); g.set_option(B.OPT_STEP_MODE, mode)
    g.prepare()
    g.set_state(B.FIELD_V, wl.initial_v())
    start, ns, bin_steps = 1000, 40, 20
    g.enable_statistics(start_step=start, bin_steps=bin_steps, sample_per_pop=ns, max_bins=4096)
    with pytest.raises(B.NgError):
        g.enable_statistics()
    g.simulate(2500); g.simulate(3500)                       # two calls: the accumulators carry over
    end = 6000
    steps, ids = g.get_spikes()
    assert steps.size > 2000
    rate, cv = g.rate_cv()
    o_rate, o_cv = S.rate_cv(steps, ids, N, start, end, 0.1)
    assert np.allclose(rate, o_rate, rtol=1e-6, atol=0)
    assert np.array_equal(np.isnan(cv), np.isnan(o_cv)) and np.count_nonzero(~np.isnan(cv)) > 100
    ok = ~np.isnan(o_cv)
    assert np.allclose(cv[ok], o_cv[ok], rtol=1e-5, atol=1e-6)
    n_bins = (end - start) // bin_steps
    for p, (first, n_pop) in enumerate(wl.pop_ranges()):
        sample = list(range(first, first + min(ns, n_pop)))
        Cg = g.correlations(p)
        Co = S.correlation(S.binned_trains(steps, ids, sample, start, n_bins, bin_steps))
        assert Cg.shape == Co.shape and np.array_equal(np.isnan(Cg), np.isnan(Co))
        okc = ~np.isnan(Co)
        assert np.allclose(Cg[okc], Co[okc], atol=2e-6)
        assert np.allclose(np.diag(Cg)[~np.isnan(np.diag(Cg))], 1.0, atol=1e-6)
    g.close()
