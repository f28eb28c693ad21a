"""Test-side helpers: build the same seeded workload on the oracle and on the CUDA path, canonicalise
connectivity, and run the lockstep protocol of DESIGN.md.  Nothing here is used by the product."""
from __future__ import annotations

import numpy as np


def make_pair(wl, oracle_mod, debug_input=True, record=True, pre_options=None, **sim_kw):
    """(oracle, gpu sim) for workload `wl`, both prepared, same fp32 initial V.  `pre_options`: {option: value} set
    before ng_prepare (the spike-buffer backend, delivery kernel 4, must be chosen there)."""
    from paper_2007_14236_b200 import binding as B
    o = oracle_mod.Oracle(0.1, wl.ring_slots, wl.seed)
    wl.apply(o)
    o.prepare()
    g = B.Sim(0.1, wl.ring_slots, wl.seed, record_spikes=record, debug_input=debug_input, **sim_kw)
    wl.apply(g)
    for opt, val in (pre_options or {}).items():
        g.set_option(opt, val)
    g.prepare()
    if not wl.bypass_neurons:
        v0 = wl.initial_v()
        o.set_state(oracle_mod.FIELD_V, v0.astype(np.float64))
        g.set_state(B.FIELD_V, v0)
    return o, g


def gpu_canonical(g):
    """GPU connection structure as (src, tgt, wbits, delay) sorted by (src, delay, tgt, wbits), plus row lengths."""
    ro = g.row_offsets()
    tgt, w, d = g.records()
    lens = np.diff(ro)
    src = np.repeat(np.arange(lens.size, dtype=np.int32), lens)
    keep = tgt >= 0
    src, tgt, w, d = src[keep], tgt[keep], w[keep], d[keep]
    wb = w.view(np.uint32)
    order = np.lexsort((wb, tgt, d, src))
    return src[order], tgt[order], wb[order], d[order], ro


def oracle_canonical(o):
    src, tgt, w, d, ro = o.get_connections()
    wb = w.view(np.uint32)
    order = np.lexsort((wb, tgt, d, src))
    return src[order], tgt[order], wb[order], d[order], ro


def check_structure(g, o, max_weight_ulp_mismatch=0):
    """Connectivity and delivery indexing bit-exact (C18); returns the number of 1-ulp weight mismatches."""
    gs, gt, gw, gd, gro = gpu_canonical(g)
    os_, ot, ow, od, oro = oracle_canonical(o)
    assert gs.size == os_.size == o.n_connections
    assert np.array_equal(gs, os_), "sources differ"
    assert np.array_equal(gd, od), "delays differ"
    assert np.array_equal(gt, ot), "targets differ"
    # out-degree per source and padded row offsets
    deg = np.diff(oro)
    assert np.array_equal(np.diff(gro), (deg + 3) // 4 * 4)
    # group offsets = prefix sums of the per-(source, delay) histogram, groups in increasing delay order
    D = g.D
    go = g.group_offsets()
    hist = np.zeros((deg.size, D + 1), np.int64)
    np.add.at(hist, (os_, od.astype(np.int64)), 1)
    expect = np.cumsum(hist, axis=1)
    assert np.array_equal(go.astype(np.int64), expect), "group offsets differ"
    bad = np.nonzero(gw != ow)[0]
    if bad.size:
        # DESIGN.md C4: device and glibc log/sincos may differ in the last bit -> at most 1 fp32 ulp, rare
        gwf, owf = gw[bad].view(np.float32), ow[bad].view(np.float32)
        assert np.all(np.abs(gw[bad].astype(np.int64) - ow[bad].astype(np.int64)) <= 1), (gwf[:5], owf[:5])
    assert bad.size <= max_weight_ulp_mismatch, f"{bad.size} weight mismatches"
    return int(bad.size)


def raw_layout_ok(g):
    """Rows are delay-grouped in place: record delays inside each row are non-decreasing and match the group table;
    padding only at row ends; inside a group records are ordered by (target, weight bits)."""
    ro = g.row_offsets()
    go = g.group_offsets().astype(np.int64)
    tgt, w, d = g.records()
    N, D = go.shape[0], go.shape[1] - 1
    deg = go[:, D]
    lens = np.diff(ro)
    pos = np.arange(tgt.size, dtype=np.int64) - np.repeat(ro[:-1], lens)
    in_row = pos < np.repeat(deg, lens)
    assert np.all(tgt[~in_row] == -1) and np.all(tgt[in_row] >= 0)
    src = np.repeat(np.arange(N), lens)
    # delay of a record from the group table
    starts = go[src[in_row]]                              # [n_rec, D+1]
    dd = (starts[:, 1:] <= pos[in_row][:, None]).sum(axis=1) + 1
    assert np.array_equal(dd, d[in_row].astype(np.int64))
    key = (src[in_row].astype(np.int64) << 40) | (d[in_row].astype(np.int64) << 32) | tgt[in_row].astype(np.int64)
    assert np.all(np.diff(key) >= 0), "records not ordered by (source, delay, target)"
    return True


class Shadow:
    """L1-mass bookkeeping for the tolerances of DESIGN.md C12: the same delivery and decay applied to |w|."""

    def __init__(self, o, wl, oracle_mod):
        self.src, self.tgt, self.w, self.d, self.ro = o.get_connections()
        self.N, self.D = o.n_neurons, wl.ring_slots
        self.abs_ring = np.zeros((self.D, self.N))
        self.abs_I = np.zeros(self.N)
        self.P = []
        self.pop_of = np.zeros(self.N, np.int64)
        first = 0
        for pi, (_, n, params) in enumerate(wl.populations):
            self.P.append((oracle_mod.propagators(params, 0.1), params))
            self.pop_of[first:first + n] = pi
            first += n
        self.P11 = np.array([p[0][0] for p in self.P])[self.pop_of]
        self.P22 = np.array([p[0][1] for p in self.P])[self.pop_of]
        self.P21 = np.array([p[0][2] for p in self.P])[self.pop_of]
        self.E_L = np.array([p[1]["E_L"] for p in self.P])[self.pop_of]
        self.V_th = np.array([p[1]["V_th"] for p in self.P])[self.pop_of]
        self.w_ext = np.array([abs(p[1]["poisson_weight"]) for p in self.P])[self.pop_of]

    def consume(self, n):
        a = self.abs_ring[n % self.D].copy()
        self.abs_ring[n % self.D] = 0.0
        return a

    def deliver(self, n, spikes):
        for j in spikes:
            lo, hi = self.ro[j], self.ro[j + 1]
            np.add.at(self.abs_ring, ((n + self.d[lo:hi].astype(np.int64)) % self.D, self.tgt[lo:hi]), np.abs(self.w[lo:hi]))
