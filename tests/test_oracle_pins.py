"""Pins for the CPU oracle (oracle/oracle.cpp) against things other than itself.

Each test names the passage of PAPER.md (or the DESIGN.md reading) it pins.  None of them needs a GPU.
"""
import math
import os

import numpy as np
import pytest
import scipy.linalg
import scipy.stats

from paper_2007_14236_b200 import workloads as W

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")
LIF = dict(W.LIF, poisson_rate_hz=0.0, poisson_weight=0.0)


# ------------------------------------------------------------------ Philox (reading C1)
def test_philox_known_answers(oracle_mod):
    rows = [l.split() for l in open(os.path.join(GOLDEN, "philox4x32_10_kat.txt")) if l.strip() and l[0] != "#"]
    assert len(rows) == 3
    for r in rows:
        v = [int(x, 16) for x in r]
        out = oracle_mod.philox4x32_10(v[4], v[5], v[0:4])
        assert [int(x) for x in out] == v[6:10]


def test_philox_counter_sensitivity(oracle_mod):
    # every counter word and both key words must enter the output (a dropped operand would collide)
    base = oracle_mod.philox4x32_10(1, 2, [3, 4, 5, 6])
    seen = {tuple(base)}
    for i in range(4):
        c = [3, 4, 5, 6]
        c[i] += 1
        seen.add(tuple(oracle_mod.philox4x32_10(1, 2, c)))
    seen.add(tuple(oracle_mod.philox4x32_10(2, 2, [3, 4, 5, 6])))
    seen.add(tuple(oracle_mod.philox4x32_10(1, 3, [3, 4, 5, 6])))
    assert len(seen) == 7


# ------------------------------------------------------------------ propagators (Eqs. 1-2 at 93-102)
def test_propagators_equal_matrix_exponential(oracle_mod):
    for h, tau_m, tau_s, C in [(0.1, 10.0, 0.5, 250.0), (0.1, 20.0, 2.0, 100.0), (1.0, 10.0, 0.5, 250.0)]:
        p = dict(LIF, tau_m=tau_m, tau_syn=tau_s, C_m=C)
        P11, P22, P21, P20 = oracle_mod.propagators(p, h)
        # x = (I, V-E_L, 1)^T with a unit constant current in the third slot: dx/dt = A x
        A = np.array([[-1 / tau_s, 0, 0], [1 / C, -1 / tau_m, 1 / C], [0, 0, 0]])
        E = scipy.linalg.expm(A * h)
        assert E[0, 0] == pytest.approx(P11, rel=1e-13)
        assert E[1, 1] == pytest.approx(P22, rel=1e-13)
        assert E[1, 0] == pytest.approx(P21, rel=1e-11)
        assert E[1, 2] == pytest.approx(P20, rel=1e-11)
        assert E[0, 1] == 0.0


def test_propagators_printed_values_and_semigroup(oracle_mod):
    # values evaluated in fp64 for the config-0 neuron
    P11, P22, P21, P20 = oracle_mod.propagators(LIF, 0.1)
    assert P11 == pytest.approx(0.818730753077982, rel=1e-14)
    assert P22 == pytest.approx(0.990049833749168, rel=1e-14)
    assert P21 == pytest.approx(3.606717487814448e-4, rel=1e-12)
    assert P20 == pytest.approx(3.9800665003327575e-4, rel=1e-12)
    Q11, Q22, Q21, Q20 = oracle_mod.propagators(LIF, 0.2)
    assert Q11 == pytest.approx(P11 * P11, rel=1e-14)
    assert Q22 == pytest.approx(P22 * P22, rel=1e-14)
    assert Q21 == pytest.approx(P22 * P21 + P21 * P11, rel=1e-12)
    assert Q20 == pytest.approx(P20 * (1 + P22), rel=1e-12)


# ------------------------------------------------------------------ single PSC response + delay convention (C10, C13)
def _two_neuron(oracle_mod, delay, w=W.W_E, D=20):
    o = oracle_mod.Oracle(0.1, D, 7)
    a = o.create_population(1, LIF)
    b = o.create_population(1, LIF)
    o.connect_fixed_indegree(a, 1, b, 1, 1, ("const", w), ("const", delay))
    o.prepare()
    return o


@pytest.mark.parametrize("delay", [1, 3, 20])
def test_psp_closed_form_on_grid(oracle_mod, delay):
    o = _two_neuron(oracle_mod, delay)
    o.set_state(oracle_mod.FIELD_V, [-40.0, -65.0])      # neuron 0 starts above threshold: spikes in step 0
    tau_m, tau_s, C = 10.0, 0.5, 250.0
    w = float(np.float32(W.W_E))                           # connection weights are fp32 quantities (record layout)
    A = w * tau_m * tau_s / (C * (tau_m - tau_s))
    vs, cur = [], []
    for n in range(delay + 60):
        o.simulate(1)
        vs.append(o.get_state(oracle_mod.FIELD_V)[1] + 65.0)
        cur.append(o.get_state(oracle_mod.FIELD_I_SYN)[1])
    st, ids = o.get_spikes()
    assert list(st) == [0] and list(ids) == [0]
    # spike found in step 0 has time t_1 = h; delay d => I jumps by exactly w at t_{1+d}, i.e. after step d
    for n in range(delay):
        assert cur[n] == 0.0 and vs[n] == 0.0
    assert cur[delay] == pytest.approx(w, rel=1e-15)
    assert vs[delay] == 0.0                               # V uses the current *before* its update (C11)
    for k in range(1, 60):
        t = 0.1 * k
        exact = A * (math.exp(-t / tau_m) - math.exp(-t / tau_s))
        assert vs[delay + k] == pytest.approx(exact, rel=1e-11)
    # first grid values and the 0.15 mV PSP amplitude the 87.8 pA weight is designed to give
    assert vs[delay + 1] == pytest.approx(0.0316669795430, rel=1e-7)
    assert vs[delay + 5] == pytest.approx(0.1078276390238, rel=1e-7)
    t_peak = math.log(tau_m / tau_s) * tau_m * tau_s / (tau_m - tau_s)
    assert t_peak == pytest.approx(1.5767012, rel=1e-6)
    assert max(vs) == pytest.approx(0.1499854908, rel=2e-4)
    assert int(np.argmax(vs)) - delay == 16


def test_inhibitory_sign(oracle_mod):
    o = _two_neuron(oracle_mod, 2, w=-351.2)
    o.set_state(oracle_mod.FIELD_V, [-40.0, -65.0])
    o.simulate(10)
    assert o.get_state(oracle_mod.FIELD_V)[1] < -65.0


# ------------------------------------------------------------------ threshold / reset / refractoriness (C11)
def test_refractory_grid_isi_closed_form(oracle_mod):
    I_e = 500.0
    o = oracle_mod.Oracle(0.1, 20, 1)
    o.create_population(1, dict(LIF, I_e=I_e))
    o.prepare()
    o.simulate(2000)
    st, _ = o.get_spikes()
    R = 10.0 / 250.0
    t_star = 10.0 * math.log(R * I_e / (R * I_e - 15.0))          # charging time from reset (=E_L) to threshold
    m_star = math.ceil(t_star / 0.1)
    assert abs(t_star / 0.1 - round(t_star / 0.1)) > 1e-6
    isi = np.diff(st)
    assert len(st) >= 10
    assert st[0] == m_star - 1                                     # first spike: m_star free updates from V = E_L
    assert np.all(isi == 20 + m_star)                              # 2 ms held + charging, on the grid


def test_refractory_clamps_v_but_current_integrates(oracle_mod):
    o = _two_neuron(oracle_mod, 1)
    # neuron 1 is made refractory by hand; a PSC arriving meanwhile must charge I but not V
    o.set_state(oracle_mod.FIELD_V, [-40.0, -65.0])
    o.set_state(oracle_mod.FIELD_REFR, [0, 5])
    o.simulate(2)
    assert o.get_state(oracle_mod.FIELD_I_SYN)[1] == pytest.approx(W.W_E, rel=1e-7)
    assert o.get_state(oracle_mod.FIELD_V)[1] == -65.0
    assert o.get_state(oracle_mod.FIELD_REFR)[1] == 3
    o.simulate(3)
    assert o.get_state(oracle_mod.FIELD_REFR)[1] == 0
    assert o.get_state(oracle_mod.FIELD_V)[1] == -65.0
    o.simulate(1)
    assert o.get_state(oracle_mod.FIELD_V)[1] > -65.0
    # threshold test is V >= V_th and reset lands exactly on V_reset
    o2 = oracle_mod.Oracle(0.1, 20, 1)
    o2.create_population(1, dict(LIF, V_reset=-70.0))
    o2.prepare()
    o2.set_state(oracle_mod.FIELD_V, [-65.0 + (-50.0 + 65.0) / 0.990049833749168 + 1e-9])
    o2.simulate(1)
    assert list(o2.get_spikes()[1]) == [0]
    assert o2.get_state(oracle_mod.FIELD_V)[0] == -70.0
    assert o2.get_state(oracle_mod.FIELD_REFR)[0] == 20


# ------------------------------------------------------------------ Poisson drive (C7)
@pytest.mark.parametrize("lam", [0.08, 0.8, 1.2, 1.28, 1.52, 1.6, 1.68, 2.32, 7.5])
def test_poisson_table_is_integer_cdf(oracle_mod, lam):
    T = oracle_mod.poisson_table(lam).astype(np.float64)
    cdf = scipy.stats.poisson.cdf(np.arange(len(T)), lam) * 2.0 ** 32
    assert T[-1] == 2 ** 32 - 1
    assert np.all(np.diff(T) >= 0)
    assert np.all(np.abs(T[:-1] - np.floor(cdf[:-1])) <= 4)       # fp64 summation-order slack only
    assert scipy.stats.poisson.sf(len(T) - 1, lam) < 2.0 ** -31        # truncated tail is below one table unit


def test_poisson_counts_follow_the_distribution(oracle_mod):
    lam = 1.28
    o = oracle_mod.Oracle(0.1, 20, 99)
    o.create_population(200, dict(LIF, poisson_rate_hz=lam / 1e-4, poisson_weight=1.0))
    o.prepare()
    ks = np.array([o.poisson_count(i, n) for i in range(200) for n in range(1000)])
    m = len(ks)
    assert ks.mean() == pytest.approx(lam, abs=5 * math.sqrt(lam / m))
    assert ks.var() == pytest.approx(lam, rel=0.03)
    obs = np.bincount(ks, minlength=8)[:8].astype(float)
    obs[7] += m - obs.sum()
    exp = scipy.stats.poisson.pmf(np.arange(8), lam) * m
    exp[7] += m - exp.sum()
    assert scipy.stats.chisquare(obs, exp).pvalue > 1e-4
    # counts of different neurons / steps are uncorrelated
    k2 = ks.reshape(200, 1000)
    assert abs(np.corrcoef(k2[0], k2[1])[0, 1]) < 0.15
    assert abs(np.corrcoef(k2[:, 0], k2[:, 1])[0, 1]) < 0.3


def test_poisson_driven_membrane_matches_campbell(oracle_mod):
    # isolated neurons, threshold disabled: shot-noise mean and variance (Campbell's theorem) of Eqs. (1)-(2)
    nu, w = 800.0, W.W_E
    o = oracle_mod.Oracle(0.1, 20, 5)
    o.create_population(400, dict(LIF, V_th=1e9, poisson_rate_hz=nu, poisson_weight=w))
    o.prepare()
    o.simulate(1500, record=False)                                  # 15 tau_m of burn-in
    samples = []
    for _ in range(40):
        o.simulate(250, record=False)
        samples.append(o.get_state(oracle_mod.FIELD_V) + 65.0)
    v = np.concatenate(samples)
    tau_m, tau_s, C = 10.0, 0.5, 250.0
    mean = (tau_m / C) * w * nu * 1e-3 * tau_s
    A = w * tau_m * tau_s / (C * (tau_m - tau_s))
    var = nu * 1e-3 * A * A * (tau_m / 2 + tau_s / 2 - 2 * tau_m * tau_s / (tau_m + tau_s))
    assert mean == pytest.approx(1.4048, rel=1e-4)
    assert math.sqrt(var) == pytest.approx(0.3427, rel=1e-3)
    assert v.mean() == pytest.approx(mean, rel=0.01)
    assert v.std() == pytest.approx(math.sqrt(var), rel=0.03)


# ------------------------------------------------------------------ connection builder (C1-C6, C18)
def test_fixed_indegree_structure_cfg0(oracle_mod):
    wl = W.brunel_tiny()
    o = wl.apply(oracle_mod.Oracle(0.1, wl.ring_slots, wl.seed))
    o.prepare()
    src, tgt, w, d, ro = o.get_connections()
    assert len(src) == wl.n_connections == 100_000
    # exactly K records per target per call
    is_e = src < 800
    assert np.all(np.bincount(tgt[is_e], minlength=1000) == 80)
    assert np.all(np.bincount(tgt[~is_e], minlength=1000) == 20)
    assert np.all(w[is_e] == np.float32(87.8)) and np.all(w[~is_e] == np.float32(-351.2))
    # row offsets are the prefix sum of the out-degree histogram; rows ordered by (delay, tgt)
    assert np.array_equal(ro, np.concatenate([[0], np.cumsum(np.bincount(src, minlength=1000))]))
    assert np.all(np.diff(src) >= 0)
    same = np.diff(src) == 0
    assert np.all(np.diff(d.astype(int))[same] >= 0)
    assert d.min() == 1 and d.max() == 20
    # uniformity of sources within each pool and of delays (chi-square against the flat law)
    assert scipy.stats.chisquare(np.bincount(src[is_e], minlength=800)[:800]).pvalue > 1e-4
    assert scipy.stats.chisquare(np.bincount(src[~is_e] - 800, minlength=200)).pvalue > 1e-4
    assert scipy.stats.chisquare(np.bincount(d, minlength=21)[1:]).pvalue > 1e-4
    # source index and delay come from different Philox words: no correlation
    assert abs(np.corrcoef(src[is_e], d[is_e])[0, 1]) < 0.02
    # O(1) regeneration of single draws lands in the list
    key = set(zip(src.tolist(), tgt.tolist(), d.tolist()))
    for call, e, k in [(0, 0, 0), (0, 799, 79), (1, 800, 5), (2, 17, 19), (3, 999, 0)]:
        s_, t_, d_, w_ = o.draw_connection(call, e, k)
        assert t_ == e and (s_, t_, d_) in key


def test_fixed_outdegree_structure(oracle_mod):
    wl = W.delivery_microbench(n=500, K=40, fraction=0.05)
    o = wl.apply(oracle_mod.Oracle(0.1, 64, 3))
    o.prepare()
    src, tgt, w, d, ro = o.get_connections()
    assert np.all(np.bincount(src, minlength=500) == 40)
    assert np.array_equal(ro, np.arange(501) * 40)
    assert d.min() >= 1 and d.max() <= 64 and len(np.unique(d)) == 64
    assert scipy.stats.chisquare(np.bincount(tgt, minlength=500)).pvalue > 1e-4


def test_normal_weights_and_delays(oracle_mod):
    o = oracle_mod.Oracle(0.1, 64, 12)
    a = o.create_population(300, LIF)
    b = o.create_population(300, LIF)
    o.connect_fixed_indegree(a, 300, b, 300, 400, ("normal", 87.8, 8.78), ("normal", 15.0, 7.5, 1, 64))
    o.connect_fixed_indegree(b, 300, a, 300, 300, ("normal", -351.2, 35.12), ("normal", 7.5, 3.75, 1, 64))
    o.prepare()
    src, tgt, w, d, _ = o.get_connections()
    e = src < 300
    z = (w[e].astype(np.float64) - 87.8) / 8.78
    assert scipy.stats.kstest(z, "norm").pvalue > 1e-4
    zi = (w[~e].astype(np.float64) + 351.2) / 35.12
    assert scipy.stats.kstest(zi, "norm").pvalue > 1e-4
    assert np.all(w[~e] < 0)
    # delays: round-half-up of N(15, 7.5) clipped to [1, 64]  (reading C5)
    for mask, mu, sd in [(e, 15.0, 7.5), (~e, 7.5, 3.75)]:
        dd = d[mask].astype(int)
        edges = np.arange(1, 65) + 0.5                     # d = floor(x + 0.5): d=k for x in [k-.5, k+.5)
        cdf = scipy.stats.norm.cdf(edges, mu, sd)
        p = np.diff(np.concatenate([[0.0], cdf[:-1], [1.0]]))
        obs = np.bincount(dd, minlength=65)[1:]
        keep = p * len(dd) > 5
        pk = np.append(p[keep], p[~keep].sum())
        ok = np.append(obs[keep], obs[~keep].sum()).astype(float)
        assert scipy.stats.chisquare(ok, pk / pk.sum() * ok.sum()).pvalue > 1e-4
        assert dd.min() >= 1
    # the two Box-Muller branches are independent
    assert abs(np.corrcoef(z, d[e])[0, 1]) < 0.02


# ------------------------------------------------------------------ delivery: plain definition by brute force (<= 50 neurons)
def _small_net(oracle_mod, D, seed=4, N=40):
    o = oracle_mod.Oracle(0.1, D, seed)
    p = dict(LIF, poisson_rate_hz=15000.0, poisson_weight=W.W_E)
    a = o.create_population(N - 10, p)
    b = o.create_population(10, p)
    dl = ("uniform_int", 1, 12)
    o.connect_fixed_indegree(a, N - 10, a, N - 10, 8, ("normal", 87.8, 8.78), dl)
    o.connect_fixed_indegree(a, N - 10, b, 10, 8, ("const", 87.8), ("normal", 6.0, 3.0, 1, 12))
    o.connect_fixed_indegree(b, 10, a, N - 10, 4, ("const", -351.2), dl)
    o.connect_fixed_outdegree(b, 10, b, 10, 3, ("const", -351.2), ("const", 12))
    o.prepare()
    g = np.random.Generator(np.random.PCG64(seed))
    o.set_state(oracle_mod.FIELD_V, g.normal(-56.0, 6.0, N))
    return o


def test_delivery_equals_plain_definition_bruteforce(oracle_mod):
    D, N, steps = 12, 40, 300
    o = _small_net(oracle_mod, D)
    src, tgt, w, d, ro = o.get_connections()
    Wd = np.zeros((D + 1, N, N))                               # dense W[d][i][j]
    np.add.at(Wd, (d.astype(int), tgt, src), w.astype(np.float64))
    S = np.zeros((steps, N))                                   # spike history S_j(m)
    row_sum = np.array([w[ro[j]:ro[j + 1]].astype(np.float64).sum() for j in range(N)])
    total_spikes = 0
    for n in range(steps):
        plane = o.get_state(oracle_mod.FIELD_RING, N, (n % D) * N)
        brute = np.zeros(N)
        for dd in range(1, D + 1):
            if n - dd >= 0:
                brute += Wd[dd] @ S[n - dd]
        assert np.allclose(plane, brute, rtol=1e-12, atol=1e-9)
        ring_before = o.get_state(oracle_mod.FIELD_RING)
        o.simulate(1)
        ring_after = o.get_state(oracle_mod.FIELD_RING)
        ids = o.last_spikes()
        S[n, ids] = 1.0
        total_spikes += len(ids)
        # invariant: what the step added to the ring is the outgoing weight of the spiking sources
        added = ring_after.sum() - (ring_before.sum() - plane.sum())
        assert added == pytest.approx(row_sum[ids].sum(), abs=1e-6)
        assert np.all(ring_after.reshape(D, N)[n % D] == 0.0) or D in d[np.isin(src, ids)]
    assert total_spikes > 50                                    # the test exercised real traffic
    st, ids = o.get_spikes()
    assert len(st) == total_spikes and np.all(np.diff(st) >= 0)


def test_results_independent_of_ring_depth(oracle_mod):
    spikes = []
    for D in (12, 13, 31):
        o = _small_net(oracle_mod, D)
        o.simulate(400)
        spikes.append(o.get_spikes())
    for s in spikes[1:]:
        assert np.array_equal(s[0], spikes[0][0]) and np.array_equal(s[1], spikes[0][1])
    assert len(spikes[0][0]) > 50


def test_delay_outside_ring_is_rejected(oracle_mod):
    o = oracle_mod.Oracle(0.1, 8, 1)
    a = o.create_population(4, LIF)
    o.connect_fixed_indegree(a, 4, a, 4, 2, ("const", 1.0), ("const", 9))
    with pytest.raises(RuntimeError):
        o.prepare()


def test_bypass_mode_injection_rate_and_delivery(oracle_mod):
    wl = W.delivery_microbench(n=2000, K=30, fraction=0.05)
    o = wl.apply(oracle_mod.Oracle(0.1, 64, 8))
    o.prepare()
    src, tgt, w, d, ro = o.get_connections()
    counts = []
    for n in range(100):
        before = o.get_state(oracle_mod.FIELD_RING).sum()
        plane = o.get_state(oracle_mod.FIELD_RING, 2000, (n % 64) * 2000).sum()
        o.simulate(1)
        ids = o.last_spikes()
        counts.append(len(ids))
        exp = sum(w[ro[j]:ro[j + 1]].astype(np.float64).sum() for j in ids)
        assert o.get_state(oracle_mod.FIELD_RING).sum() - (before - plane) == pytest.approx(exp, abs=1e-6)
    tot = sum(counts)
    assert tot == pytest.approx(0.05 * 2000 * 100, abs=5 * math.sqrt(0.05 * 0.95 * 2000 * 100))
    assert o.n_events == tot * 30


# ------------------------------------------------------------------ workload recipe pins (C6, C15)
def test_microcircuit_recipe_matches_paper_scale():
    vals = {}
    for l in open(os.path.join(GOLDEN, "paper_values.txt")):
        l = l.split("#")[0].split()
        if len(l) == 2:
            vals[l[0]] = float(l[1])
    full = W.microcircuit(1)
    assert full.n_neurons == 77169
    assert abs(full.n_neurons - vals["microcircuit_neurons_approx"]) / vals["microcircuit_neurons_approx"] < 0.01
    assert full.n_connections == 298_905_266
    assert abs(full.n_connections - vals["microcircuit_connections_approx"]) < 0.01 * vals["microcircuit_connections_approx"]
    assert len(full.populations) == vals["microcircuit_populations"]
    # reading C6-B: literal in-degrees follow from BASELINE.json's probabilities
    for t in range(8):
        for s in range(8):
            p = W.PD_CONN_PROB[t][s]
            if p == 0:
                assert W.PD_INDEGREE[t][s] == 0
                continue
            k_tot = round(math.log(1 - p) / math.log(1 - 1 / (W.PD_SIZES[s] * W.PD_SIZES[t])))
            assert W.PD_INDEGREE[t][s] == round(k_tot / W.PD_SIZES[t])
    tenth = W.microcircuit(10)
    assert [p[1] for p in tenth.populations] == [2068, 583, 2192, 548, 485, 107, 1440, 295]
    assert tenth.n_connections == 29_892_043
    assert W.balanced_large().n_connections == 10 ** 9
    assert W.brunel_tiny().n_connections == 10 ** 5
