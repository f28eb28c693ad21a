"""Pins of the AdEx part of the oracle (oracle/oracle_adex.hpp) against things other than itself: scipy's stiff ODE
solvers on the single-neuron protocol the paper itself validates with (one AdEx neuron, 700 pA), the
closed-form alpha conductance, hand-evaluated right-hand sides, and brute force of the two-port delivery."""
import numpy as np
import pytest
from scipy.integrate import solve_ivp

from paper_2007_14236_b200 import workloads as W


def params(**over):
    p = dict(W.ADEX)
    p.update(over)
    return p


def scipy_rhs(p, clamp=True):
    def f(t, y):
        V = min(y[0], p["V_peak"]) if clamp else y[0]      # the clamp only matters beyond the spike event
        return [(-p["g_L"] * (V - p["E_L"]) + p["g_L"] * p["Delta_T"] * np.exp((V - p["V_T"]) / p["Delta_T"])
                 + y[2] * (p["E_ex"] - V) + y[4] * (p["E_in"] - V) - y[1] + p["I_e"]) / p["C_m"],
                (p["a"] * (V - p["E_L"]) - y[1]) / p["tau_w"],
                -y[2] / p["tau_syn"] + y[3], -y[3] / p["tau_syn"], -y[4] / p["tau_syn"] + y[5], -y[5] / p["tau_syn"]]
    return f


def test_rhs_hand_values(oracle_mod):
    p = params(I_e=100.0)
    y = np.array([-55.0, 20.0, 1.5, 0.3, 0.7, -0.1])
    f = oracle_mod.adex_rhs(p, y)
    dV = (-30.0 * (-55.0 + 70.6) + 30.0 * 2.0 * np.exp((-55.0 + 50.4) / 2.0) + 1.5 * (0.0 + 55.0) + 0.7 * (-85.0 + 55.0)
          - 20.0 + 100.0) / 281.0                                   # Eq. (3) with reading C21, typed out by hand
    assert f[0] == pytest.approx(dV, rel=1e-14)
    assert f[1] == pytest.approx((4.0 * (-55.0 + 70.6) - 20.0) / 144.0, rel=1e-14)      # Eq. (5)
    assert f[2] == pytest.approx(-1.5 + 0.3) and f[3] == pytest.approx(-0.3)
    assert f[4] == pytest.approx(-0.7 - 0.1) and f[5] == pytest.approx(0.1)
    # C21: an excitatory conductance depolarises, an inhibitory one hyperpolarises (at rest, between the reversals)
    rest = np.array([-70.6, 0, 0, 0, 0, 0.0])
    f0 = oracle_mod.adex_rhs(params(), rest)[0]
    assert oracle_mod.adex_rhs(params(), rest + [0, 0, 1, 0, 0, 0])[0] > f0 > oracle_mod.adex_rhs(params(), rest + [0, 0, 0, 0, 1, 0])[0]
    # exponential clamped at V_peak (C24)
    assert oracle_mod.adex_rhs(params(), [50.0, 0, 0, 0, 0, 0])[0] == oracle_mod.adex_rhs(params(), [0.0, 0, 0, 0, 0, 0])[0]


def test_alpha_conductance_closed_form(oracle_mod):
    """C22: y jumps by W e / tau; g(t) = W (t / tau) exp(1 - t / tau), peak W at t = tau."""
    p = params()
    Wn = 0.05
    y = np.array([-70.6, 0, 0, Wn * np.e / p["tau_syn"], 0, 0.35 * np.e / p["tau_syn"]]); h = 0.1
    g_ex, g_in = [], []
    for k in range(60):
        y, h, _ = oracle_mod.adex_step(p, y, h, 0.1)
        g_ex.append(y[2]); g_in.append(y[4])
    t = 0.1 * np.arange(1, 61)
    assert np.allclose(g_ex, Wn * t * np.exp(1 - t), atol=2e-5)
    assert np.allclose(g_in, 0.35 * t * np.exp(1 - t), atol=1e-4)
    assert abs(max(g_ex) - Wn) < 1e-4 and int(np.argmax(g_ex)) == 9          # peak W one tau after the spike


def test_single_neuron_700pA_against_scipy(oracle_mod):
    """PAPER.md:252 protocol.  Reference: scipy DOP853 (rtol 1e-11) with an event at V_peak, reset by hand."""
    p = params(I_e=700.0)
    f = scipy_rhs(p, clamp=False)
    ev = lambda t, y: y[0] - p["V_peak"]
    ev.terminal = True; ev.direction = 1
    T = 300.0
    t0, y0, ref_spikes, segs = 0.0, [p["E_L"], 0, 0, 0, 0, 0], [], []
    while t0 < T:
        sol = solve_ivp(f, (t0, T), y0, method="DOP853", rtol=1e-11, atol=1e-12, events=ev, dense_output=True)
        segs.append((t0, sol.t[-1], sol.sol))
        if sol.status == 1:
            t0 = sol.t_events[0][0]; ref_spikes.append(t0)
            y0 = sol.y[:, -1].copy(); y0[0] = p["V_reset"]; y0[1] += p["b"]
        else:
            break
    y = np.array([p["E_L"], 0, 0, 0, 0, 0.0]); h = 0.1
    spikes, Vs = [], []
    for k in range(int(T / 0.1)):
        y, h, s = oracle_mod.adex_step(p, y, h, 0.1)
        Vs.append(y[0])
        if s:
            spikes.append(k)
    assert len(ref_spikes) >= 4 and len(spikes) == len(ref_spikes)
    # a spike is found in the step that contains the reference crossing (resets happen on sub-step boundaries, so the
    # trajectories after the first spike are shifted by less than one sub-step)
    assert all(abs(k - int(tr / 0.1)) <= 1 for k, tr in zip(spikes, ref_spikes))
    # before the first spike the trajectory is the same ODE: compare away from the upswing
    k1 = spikes[0]
    tg = 0.1 * np.arange(1, k1 - 5)
    ref = segs[0][2](tg)[0]
    sel = ref < -45.0
    assert np.max(np.abs(np.array(Vs[:k1 - 6]) - ref)[sel]) < 2e-3
    # adaptation: inter-spike intervals grow (w accumulates b per spike)
    assert np.all(np.diff(np.diff(spikes)) > 0)


def reference_spike_times(p, T):
    """Spike times of one AdEx neuron under a constant current: scipy DOP853 (rtol 1e-11) with a terminal event at V_peak,
    reset (V -> V_r, w -> w + b) by hand.  Independent of the oracle's integrator, controller and sub-step floor."""
    f = scipy_rhs(p, clamp=False)
    ev = lambda t, y: y[0] - p["V_peak"]
    ev.terminal = True; ev.direction = 1
    t0, y0, out = 0.0, [p["E_L"], 0, 0, 0, 0, 0], []
    while t0 < T:
        sol = solve_ivp(f, (t0, T), y0, method="DOP853", rtol=1e-11, atol=1e-12, events=ev)
        if sol.status != 1:
            break
        t0 = sol.t_events[0][0]; out.append(t0)
        y0 = sol.y[:, -1].copy(); y0[0] = p["V_reset"]; y0[1] += p["b"]
    return out


def oracle_spike_steps(oracle_mod, p, T):
    y = np.array([p["E_L"], 0, 0, 0, 0, 0.0]); h = 0.1
    out = []
    for k in range(int(round(T / 0.1))):
        y, h, s = oracle_mod.adex_step(p, y, h, 0.1)
        if s:
            out.append(k)
    return out


@pytest.mark.parametrize("I_e,n_min", [(700.0, 9), (1000.0, 30)])
def test_spike_steps_and_sub_step_floor(oracle_mod, I_e, n_min):
    """Reading C23 fixes the smallest sub-step h_min of the adaptive integrator (the paper names none).  On
    the single-neuron constant-current protocol of PAPER.md:252 (700 pA; 1000 pA as a faster-firing second case), over a
    full second, EVERY spike of the oracle with the recipe's h_min = 1e-3 ms must fall in the time step that contains the
    event-located DOP853 crossing (the next step only if the crossing lies in the last tenth of its step: the integrator's
    own phase error is a few 1e-3 ms) and the lag must not accumulate — spike steps and inter-spike intervals, not only the
    subthreshold trace.  The looser floor 1e-2 ms (used for speed during round 1) does not meet this: sub-steps at the
    floor are accepted unconditionally, each spike is found ~0.01 ms late and the lag grows to whole steps; asserted here
    so that the choice stays on evidence."""
    assert W.ADEX["h_min"] == 1e-3
    T = 1000.0
    ref = np.array(reference_spike_times(params(I_e=I_e), T))
    assert ref.size >= n_min
    ref_steps = np.floor(ref / 0.1).astype(int)
    phase = ref / 0.1 - ref_steps
    fine = np.array(oracle_spike_steps(oracle_mod, params(I_e=I_e), T))
    assert fine.size == ref.size
    lag = fine - ref_steps
    assert np.all((lag == 0) | ((lag == 1) & (phase > 0.9))), (lag, phase)
    assert np.all(np.abs(np.diff(fine) - np.diff(ref_steps)) <= 1) and lag[-1] == 0
    assert np.mean(lag == 0) >= 0.9
    coarse = np.array(oracle_spike_steps(oracle_mod, params(I_e=I_e, h_min=1e-2), T))
    assert coarse.size == ref.size
    lag_c = coarse - ref_steps
    assert lag_c.min() >= 0 and lag_c[-1] >= 1 and np.mean(lag_c >= 1) >= 0.5, lag_c          # it accumulates


def test_network_rate_is_insensitive_to_the_floor(oracle_mod):
    """The 2000-neuron balanced network of the rate pin below at both floors: same mean rate within 1 %.  (The floor moves
    single spikes by a step after tens of spikes; it does not change the population activity.)"""
    rates = {}
    for hm in (1e-3, 1e-2):
        wl = W.balanced_adex(n=2000, k_total=200, n_steps=3000, seed=5)
        wl.populations = [(name, n, dict(p, h_min=hm)) for name, n, p in wl.populations]
        o = oracle_mod.Oracle(0.1, wl.ring_slots, wl.seed)
        wl.apply(o); o.prepare()
        o.set_state(oracle_mod.FIELD_V, wl.initial_v().astype(np.float64))
        o.simulate(3000)
        st, ids = o.get_spikes()
        rates[hm] = np.sum(st >= 500) / 2000 / 0.25
    assert abs(rates[1e-3] - rates[1e-2]) <= 0.01 * rates[1e-3], rates


def test_fixed_point_and_step_size_state(oracle_mod):
    """No drive: the resting point of Eqs. (3), (5) is stationary; the sub-step size grows to the whole step."""
    p = params()
    root = solve_ivp(scipy_rhs(p), (0, 5000.0), [p["E_L"], 0, 0, 0, 0, 0], method="Radau", rtol=1e-10, atol=1e-12).y[:, -1]
    y, h = root.copy(), 0.01
    for _ in range(50):
        y, h, s = oracle_mod.adex_step(p, y, h, 0.1)
        assert not s
    assert np.allclose(y, root, atol=1e-6) and h == pytest.approx(0.1)


def test_two_port_network_brute_force(oracle_mod):
    """Delivery with receptor ports: ring[slot][port][target] equals the plain definition per port (dense brute force)."""
    wl = W.balanced_adex(n=40, k_total=10, n_steps=60, seed=4)
    o = oracle_mod.Oracle(0.1, wl.ring_slots, wl.seed)
    wl.apply(o); o.prepare()
    assert o.n_ports == 2
    N, D = 40, wl.ring_slots
    v0 = wl.initial_v(); v0[:8] = -30.0; v0[32:36] = -30.0  # a few E and I neurons start on the upswing and fire at once
    o.set_state(oracle_mod.FIELD_V, v0.astype(np.float64))
    src, tgt, w, d, ro = o.get_connections()
    port = np.where(src < 32, 0, 1)                          # E sources -> port 0, I sources -> port 1 (the recipe)
    hist = np.zeros((200, N), bool)
    seen_ports = set()
    for n in range(60):
        ring_before = o.get_state(oracle_mod.FIELD_RING).reshape(D, 2, N).copy()
        o.simulate(1)
        hist[n, o.last_spikes()] = True
        ring = o.get_state(oracle_mod.FIELD_RING).reshape(D, 2, N)
        # plain definition of every pending cell: sum over connections of w * S_src(n' - d), n' in (n, n + D]
        for npend in range(n + 1, n + 1 + D):
            exp = np.zeros((2, N))
            for c in range(src.size):
                m = npend - int(d[c])
                if 0 <= m <= n and hist[m, src[c]]:
                    exp[port[c], tgt[c]] += float(w[c])
            assert np.allclose(ring[npend % D], exp, atol=1e-12), (n, npend)
            seen_ports |= {pt for pt in (0, 1) if exp[pt].any()}
    assert hist.sum() >= 12 and seen_ports == {0, 1}


def golden():
    import os
    out = {}
    for l in open(os.path.join(os.path.dirname(__file__), "golden", "paper_values.txt")):
        l = l.split("#")[0].split()
        if len(l) == 2:
            out[l[0]] = float(l[1])
    return out


def test_recipe_matches_the_papers_tables():
    """The balanced_adex recipe carries exactly the numbers of PAPER.md Tables I and II (tests/golden/paper_values.txt)."""
    G = golden()
    for k in ("C_m", "g_L", "E_L", "V_T", "Delta_T", "tau_w", "a", "b", "V_reset", "E_ex", "E_in", "tau_syn"):
        assert W.ADEX[k] == G["adex_" + k], k
    wl = W.balanced_adex(n=1000, k_total=100)
    pe = wl.populations[0][2]
    assert pe["poisson_rate_hz"] == G["balanced_rate_poisson_hz"] and pe["poisson_weight"] == G["balanced_W_poisson"]
    assert wl.populations[1][1] * 4 == wl.populations[0][1]                      # N_in = N_ex / 4
    (_, _, _, ke, we, de, pe_), _, (_, _, _, ki, wi, di, pi_), _ = wl.calls
    assert ke == 4 * ki and we == ("const", G["balanced_W_ex"]) and wi == ("const", G["balanced_W_in"]) and (pe_, pi_) == (0, 1)
    assert de[1] * 0.1 == pytest.approx(G["balanced_delay_mean_ms"]) and de[2] * 0.1 == pytest.approx(G["balanced_delay_std_ms"])
    full = W.balanced_adex()
    assert full.n_neurons == G["balanced_max_neurons"] and full.n_connections == G["balanced_max_connections"]


def test_balanced_network_rate_near_the_papers(oracle_mod):
    """PAPER.md Table I prints the average firing rate of the balanced network: 30.7 Hz.  The paper's network sizes are
    "variable"; a 2000-neuron, 200-input instance of the same recipe must land near it (the readings C21-C25 — sign of
    Eq. (4), alpha normalisation, V_peak — each move the rate by far more than the band allowed here)."""
    wl = W.balanced_adex(n=2000, k_total=200, n_steps=3000, seed=5)
    o = oracle_mod.Oracle(0.1, wl.ring_slots, wl.seed)
    wl.apply(o); o.prepare()
    o.set_state(oracle_mod.FIELD_V, wl.initial_v().astype(np.float64))
    o.simulate(3000)
    st, ids = o.get_spikes()
    rate = np.sum(st >= 500) / 2000 / 0.25
    assert abs(rate - golden()["balanced_mean_rate_hz"]) < 0.15 * 30.7, rate
