"""The stored oracle spike counts (tests/golden/oracle_rates_*.txt, written by tests/golden/make_oracle_rates.py from
oracle/ alone) that the full-size free-running GPU parity tests compare with.  The oracle is deterministic, so a prefix
of each file is regenerated here and must match to the spike; the big files (config 2: 11 s of the full-scale
microcircuit, config 4: 1 s of the 1e6-neuron network) are checked for shape and for plausibility against the
small-scale runs."""
import os
import sys

import numpy as np
import pytest

from paper_2007_14236_b200 import workloads as W

sys.path.insert(0, os.path.join(os.path.dirname(__file__), "golden"))
import make_oracle_rates as G  # noqa: E402


@pytest.mark.parametrize("name,n_check", [("cfg0", 21), ("cfg1", 3)])
def test_golden_prefix_regenerates_exactly(oracle_mod, name, n_check):
    ws, sizes, counts = G.read_file(G.golden_path(name))
    wl = W.by_name(name)
    assert sizes == [p[1] for p in wl.populations] and ws == 1000
    again = G.window_counts(oracle_mod, wl, n_check, ws)
    assert np.array_equal(again, counts[:n_check])
    assert counts[0].sum() > 0


@pytest.mark.parametrize("name,n_windows", [("cfg1", 110), ("cfg2", 110), ("cfg4", 10)])
def test_golden_files_shape_and_rates(name, n_windows):
    path = G.golden_path(name)
    if not os.path.exists(path):
        pytest.skip(f"{path} not generated yet")
    ws, sizes, counts = G.read_file(path)
    wl = W.by_name(name)
    assert sizes == [p[1] for p in wl.populations] and counts.shape == (n_windows, len(sizes)) and ws == 1000
    skip = 10 if name != "cfg4" else 1                       # the first second is discarded
    rate = counts[skip:].sum(axis=0) / np.array(sizes) / ((n_windows - skip) * ws * 1e-4)
    assert np.all(rate > 0.05) and np.all(rate < 60.0), rate


def test_full_scale_rates_resemble_the_10_percent_network():
    """Config 2 is config 1 with ten times the neurons and the same in-degrees: its population rates are not equal (the
    10 % network has stronger correlations) but of the same order — a gross error in the stored file (a wrong population
    order, a unit slip) would show here."""
    for name in ("cfg1", "cfg2"):
        if not os.path.exists(G.golden_path(name)):
            pytest.skip("golden files not generated yet")
    _, s1, c1 = G.read_file(G.golden_path("cfg1"))
    _, s2, c2 = G.read_file(G.golden_path("cfg2"))
    r1 = c1[10:].sum(axis=0) / np.array(s1) / 10.0
    r2 = c2[10:].sum(axis=0) / np.array(s2) / 10.0
    assert np.all(r2 < 4.0 * r1 + 0.5) and np.all(r2 > 0.25 * r1 - 0.5), (r1, r2)
