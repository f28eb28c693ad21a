"""Seeded synthetic input recipes for the five BASELINE.json workloads.

This module is the ONLY thing the CUDA path's harness and the oracle's harness share.  It holds
none of the method's arithmetic: it lists populations, connect calls and distributions as plain
data and draws the initial membrane potentials with numpy.  A recipe is applied to any object that
exposes ``create_population / connect_fixed_indegree / connect_fixed_outdegree`` (the product
binding ``Sim`` and the test oracle ``Oracle`` both do).

The paper uses no dataset; the microcircuit and balanced-network *models*
are specified by BASELINE.json's numbers and DESIGN.md's readings C3-C16.  These synthetic recipes
stand in for the authors' Potjans_2014 / brunel_net scripts, which are not
reproduced here.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

# iaf_psc_exp parameters common to configs 0, 1, 2, 4 (BASELINE.json configs[0])
LIF = dict(C_m=250.0, tau_m=10.0, tau_syn=0.5, E_L=-65.0, V_th=-50.0, V_reset=-65.0, t_ref_ms=2.0, I_e=0.0)
W_E = 87.8          # pA
DT_MS = 0.1

# full-scale microcircuit population sizes, order L2/3E, L2/3I, L4E, L4I, L5E, L5I, L6E, L6I (reading C16)
PD_NAMES = ["L23E", "L23I", "L4E", "L4I", "L5E", "L5I", "L6E", "L6I"]
PD_SIZES = [20683, 5834, 21915, 5479, 4850, 1065, 14395, 2948]
PD_K_EXT = [1600, 1500, 2100, 1900, 2000, 1900, 2900, 2100]
# literal in-degree matrix, rows = target, cols = source (reading C6, pinned in tests against
# BASELINE.json's connection probabilities and the paper's "about 3e8 connections")
PD_INDEGREE = [
    [2200, 1079, 979, 468, 159, 0, 110, 0],
    [2990, 860, 704, 290, 381, 0, 61, 0],
    [160, 35, 1117, 795, 33, 0, 667, 0],
    [1481, 17, 1813, 953, 16, 0, 1608, 0],
    [2188, 375, 1136, 31, 421, 496, 297, 0],
    [1166, 159, 571, 12, 300, 404, 124, 0],
    [325, 39, 467, 92, 286, 21, 582, 752],
    [767, 6, 75, 3, 136, 9, 980, 459],
]
PD_CONN_PROB = [
    [.1009, .1689, .0437, .0818, .0323, 0, .0076, 0],
    [.1346, .1371, .0316, .0515, .0755, 0, .0042, 0],
    [.0077, .0059, .0497, .135, .0067, .0003, .0453, 0],
    [.0691, .0029, .0794, .1597, .0033, 0, .1057, 0],
    [.1004, .0622, .0505, .0057, .0831, .3726, .0204, 0],
    [.0548, .0269, .0257, .0022, .06, .3158, .0086, 0],
    [.0156, .0066, .0211, .0166, .0572, .0197, .0396, .2252],
    [.0364, .001, .0034, .0005, .0277, .008, .0658, .1443],
]


@dataclass
class Workload:
    name: str
    ring_slots: int
    seed: int
    n_steps: int
    populations: list = field(default_factory=list)      # (name, n, lif-params dict)
    calls: list = field(default_factory=list)            # (rule, src_pop, tgt_pop, K, weight dist, delay dist[, port])
    bypass_neurons: bool = False
    inject_fraction: float = 0.0
    v0_mean: float = -58.0
    v0_sd: float = 10.0                                   # reading C14: 10 is the standard deviation

    @property
    def n_neurons(self) -> int:
        return sum(p[1] for p in self.populations)

    @property
    def n_connections(self) -> int:
        tot = 0
        for rule, sp, tp, K, *_ in self.calls:
            tot += K * (self.populations[tp][1] if rule == "in" else self.populations[sp][1])
        return tot

    def pop_ranges(self):
        out, first = [], 0
        for _, n, _ in self.populations:
            out.append((first, n))
            first += n
        return out

    def apply(self, sim):
        """Create populations and issue connect calls on ``sim`` in recipe order."""
        firsts = [sim.create_population(n, params) for _, n, params in self.populations]
        rng = self.pop_ranges()
        assert firsts == [r[0] for r in rng]
        for rule, sp, tp, K, w, d, *port in self.calls:
            fn = sim.connect_fixed_indegree if rule == "in" else sim.connect_fixed_outdegree
            if port:                                     # receptor port of the targets (AdEx: 0 excitatory, 1 inhibitory)
                fn(rng[sp][0], rng[sp][1], rng[tp][0], rng[tp][1], K, w, d, port=port[0])
            else:
                fn(rng[sp][0], rng[sp][1], rng[tp][0], rng[tp][1], K, w, d)
        if self.bypass_neurons:
            sim.set_bypass(True, self.inject_fraction)
        return sim

    def initial_v(self) -> np.ndarray:
        """fp32 initial membrane potentials handed identically to both sides (reading C14)."""
        g = np.random.Generator(np.random.PCG64(self.seed + 0x5EED))
        return g.normal(self.v0_mean, self.v0_sd, self.n_neurons).astype(np.float32)


def _lif(rate_hz: float, w_ext: float = W_E, **over) -> dict:
    p = dict(LIF)
    p.update(poisson_rate_hz=rate_hz, poisson_weight=w_ext)
    p.update(over)
    return p


def brunel_tiny(n_e=800, n_i=200, k_e=80, k_i=20, g=4.0, n_steps=1000, seed=1, ext_inputs=100) -> Workload:
    """Config 0: tiny Brunel-style LIF net."""
    wl = Workload("cfg0_brunel_tiny", ring_slots=20, seed=seed, n_steps=n_steps)
    lif = _lif(8.0 * ext_inputs)
    wl.populations = [("E", n_e, lif), ("I", n_i, lif)]
    dly = ("uniform_int", 1, 20)
    wl.calls = [("in", 0, 0, k_e, ("const", W_E), dly), ("in", 0, 1, k_e, ("const", W_E), dly),
                ("in", 1, 0, k_i, ("const", -g * W_E), dly), ("in", 1, 1, k_i, ("const", -g * W_E), dly)]
    return wl


def microcircuit(scale_div: int = 1, n_steps: int = 10000, seed: int = 1, indegree_div: int = 1) -> Workload:
    """Configs 1 (scale_div=10) and 2 (scale_div=1): cortical-microcircuit-shaped LIF network.

    Population sizes are divided with the integer rule (N + scale_div//2) // scale_div (reading C15);
    in-degrees stay at full scale.  ``indegree_div`` > 1 shrinks in-degrees for small test variants only.
    """
    wl = Workload(f"cfg{'2' if scale_div == 1 else '1'}_microcircuit_div{scale_div}", ring_slots=64, seed=seed,
                  n_steps=n_steps)
    sizes = [(n + scale_div // 2) // scale_div for n in PD_SIZES]
    wl.populations = [(PD_NAMES[i], sizes[i], _lif(8.0 * PD_K_EXT[i])) for i in range(8)]
    for t in range(8):
        for s in range(8):
            K = PD_INDEGREE[t][s] // indegree_div
            if K == 0:
                continue
            exc = (s % 2 == 0)
            mean_w = W_E if exc else -4.0 * W_E
            if s == 2 and t == 0:            # L4E -> L2/3E doubled (BASELINE.json configs[1])
                mean_w *= 2.0
            w = ("normal", mean_w, 0.1 * abs(mean_w))
            # reading C5: delays in steps, E 15 +- 7.5, I 7.5 +- 3.75, clipped to [1, D]
            d = ("normal", 15.0, 7.5, 1, 64) if exc else ("normal", 7.5, 3.75, 1, 64)
            wl.calls.append(("in", s, t, K, w, d))
    return wl


def delivery_microbench(n=1_000_000, K=1000, fraction=0.01, n_steps=1000, seed=1) -> Workload:
    """Config 3: spike-delivery microbenchmark, neuron update bypassed (reading C8)."""
    wl = Workload(f"cfg3_delivery_n{n}_K{K}_f{fraction}", ring_slots=64, seed=seed, n_steps=n_steps,
                  bypass_neurons=True, inject_fraction=fraction)
    wl.populations = [("pool", n, _lif(0.0))]
    wl.calls = [("out", 0, 0, K, ("normal", W_E, 0.1 * W_E), ("uniform_int", 1, 64))]
    return wl


def balanced_large(n=1_000_000, k_total=1000, n_steps=10000, seed=1) -> Workload:
    """Config 4: large balanced E/I network, LIF stand-in for the paper's AdEx network."""
    n_e, n_i = (n * 4) // 5, n - (n * 4) // 5
    k_e, k_i = (k_total * 4) // 5, k_total - (k_total * 4) // 5
    wl = Workload(f"cfg4_balanced_n{n}_k{k_total}", ring_slots=20, seed=seed, n_steps=n_steps)
    lif = _lif(8.0 * k_total)
    wl.populations = [("E", n_e, lif), ("I", n_i, lif)]
    dly = ("uniform_int", 1, 20)
    wl.calls = [("in", 0, 0, k_e, ("const", W_E), dly), ("in", 0, 1, k_e, ("const", W_E), dly),
                ("in", 1, 0, k_i, ("const", -5.0 * W_E), dly), ("in", 1, 1, k_i, ("const", -5.0 * W_E), dly)]
    return wl


# AdEx parameters of the paper's balanced network (Table II); V_peak, t_ref and the integrator tolerances are
# not in the paper (readings C23, C24)
ADEX = dict(model="adex", C_m=281.0, g_L=30.0, E_L=-70.6, V_T=-50.4, Delta_T=2.0, tau_w=144.0, a=4.0, b=80.5, V_reset=-60.0,
            V_peak=0.0, E_ex=0.0, E_in=-85.0, tau_syn=1.0, I_e=0.0,
            tol=(2e-4, 2e-3, 2e-5, 2e-4, 2e-5, 2e-4), h_min=1e-3)


def balanced_adex(n=1_000_000, k_total=1000, n_steps=10000, seed=1) -> Workload:
    """The paper's balanced network (Table I): N_in = N_ex / 4, CI = CE / 4, W_ex = 0.05 nS, W_in = 0.35 nS
    on separate receptor ports, delays 0.5 +- 0.25 ms, Poisson drive 20 kHz x 0.37 nS, AdEx neurons of Table II."""
    n_e, n_i = (n * 4) // 5, n - (n * 4) // 5
    k_e, k_i = (k_total * 4) // 5, k_total - (k_total * 4) // 5
    wl = Workload(f"adex_balanced_n{n}_k{k_total}", ring_slots=20, seed=seed, n_steps=n_steps, v0_mean=-65.0, v0_sd=5.0)
    ax = dict(ADEX); ax.update(poisson_rate_hz=20000.0, poisson_weight=0.37)
    wl.populations = [("E", n_e, ax), ("I", n_i, ax)]
    dly = ("normal", 5.0, 2.5, 1, 20)
    wl.calls = [("in", 0, 0, k_e, ("const", 0.05), dly, 0), ("in", 0, 1, k_e, ("const", 0.05), dly, 0),
                ("in", 1, 0, k_i, ("const", 0.35), dly, 1), ("in", 1, 1, k_i, ("const", 0.35), dly, 1)]
    return wl


def by_name(name: str) -> Workload:
    return {
        "cfg0": brunel_tiny,
        "cfg1": lambda: microcircuit(10, 10000),
        "cfg2": lambda: microcircuit(1, 100000),
        "cfg3": delivery_microbench,
        "cfg4": balanced_large,
    }[name]()
