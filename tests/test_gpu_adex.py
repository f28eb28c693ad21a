"""GPU parity of the AdEx path (the model of the paper's balanced network) against the fp64 oracle.

Bars: connectivity with receptor ports bit-exact; lockstep (the GPU is fed the oracle's state, rounded to fp32, every
step): spike lists identical except neurons on the exponential upswing (V > -45 mV before the step: "away from the
peaks", logged); V within 5e-3 mV, w within 5e-2 pA, conductances within 1e-4 relative; delivered inputs per
port within 1e-5 of their L1 mass (C12); free-running population rates within 5 % (C17)."""
import numpy as np
import pytest

from paper_2007_14236_b200 import workloads as W

from helpers import make_pair

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    from paper_2007_14236_b200 import binding
    return binding


def adex_fields(B, oracle_mod):
    return [(B.FIELD_V, oracle_mod.FIELD_V), (B.FIELD_ADEX_W, oracle_mod.FIELD_W), (B.FIELD_ADEX_G_EX, oracle_mod.FIELD_G_EX),
            (B.FIELD_ADEX_Y_EX, oracle_mod.FIELD_Y_EX), (B.FIELD_ADEX_G_IN, oracle_mod.FIELD_G_IN),
            (B.FIELD_ADEX_Y_IN, oracle_mod.FIELD_Y_IN), (B.FIELD_ADEX_H, oracle_mod.FIELD_H_INT)]


def make_adex_pair(wl, oracle_mod, B, **kw):
    o, g = make_pair(wl, oracle_mod, **kw)          # make_pair feeds the same fp32 initial V to both
    return o, g


def structure_with_ports(g, o, N):
    ro = g.row_offsets(); tgt, w, d = g.records()
    src = np.repeat(np.arange(N, dtype=np.int32), np.diff(ro))
    keep = tgt >= 0
    port = tgt[keep] // N; t = tgt[keep] % N
    osrc, otgt, ow, od, _ = o.get_connections()
    go = np.lexsort((w[keep].view(np.uint32), t, d[keep], src[keep])); oo = np.lexsort((ow.view(np.uint32), otgt, od, osrc))
    assert np.array_equal(src[keep][go], osrc[oo]) and np.array_equal(t[go], otgt[oo]) and np.array_equal(d[keep][go], od[oo])
    assert np.array_equal(w[keep][go], ow[oo])
    return src[keep][go], port[go]


@pytest.mark.parametrize("mode,kernel", [(2, 3), (0, 3), (0, 1), (0, 4)])
def test_adex_lockstep(oracle_mod, B, mode, kernel):
    wl = W.balanced_adex(n=2000, k_total=100, n_steps=400, seed=3)
    o, g = make_adex_pair(wl, oracle_mod, B, pre_options={B.OPT_DELIVERY_KERNEL: kernel, B.OPT_STEP_MODE: mode})
    N, D = wl.n_neurons, wl.ring_slots
    assert o.n_ports == 2 and g.n_ports == 2
    src_sorted, port_sorted = structure_with_ports(g, o, N)
    assert np.all(port_sorted[src_sorted < 1600] == 0) and np.all(port_sorted[src_sorted >= 1600] == 1)   # E -> port 0, I -> port 1
    fields = adex_fields(B, oracle_mod)
    osrc, otgt, ow, od, oro = o.get_connections()
    oport = np.where(osrc < 1600, 0, 1)
    mass = np.zeros((D, 2, N))
    n_spk, logged = 0, []
    for n in range(400):
        st = {}
        for gf, of in fields:
            st[of] = o.get_state(of)
            g.set_state(gf, st[of].astype(np.float32))
        in_or = o.get_state(oracle_mod.FIELD_RING, 2 * N, first=(n % D) * 2 * N).reshape(2, N)
        m_in = mass[n % D].copy(); mass[n % D] = 0.0
        upswing = st[oracle_mod.FIELD_V] > -45.0
        g.simulate(1); o.simulate(1, record=False)
        gs = np.sort(g.last_spikes()); os_ = np.sort(o.last_spikes())
        diff = np.setxor1d(gs, os_)
        assert np.all(upswing[diff]), (n, diff[~upswing[diff]][:10])
        logged += diff.tolist(); n_spk += os_.size
        gin = g.get_state(B.FIELD_LAST_INPUT).astype(np.float64).reshape(2, N)
        assert np.all(np.abs(gin - in_or) <= 1e-5 * m_in + 1e-12), (n, float(np.abs(gin - in_or).max()))
        calm = ~upswing
        calm[diff] = False
        for (gf, of), tol_abs, tol_rel in zip(fields, (5e-3, 5e-2, 1e-6, 1e-5, 1e-6, 1e-5, 0), (0, 0, 1e-4, 1e-4, 1e-4, 1e-4, 0)):
            if gf == B.FIELD_ADEX_H:
                continue                                   # the controller may take different sub-steps in fp32
            a, b = g.get_state(gf).astype(np.float64), o.get_state(of)
            assert np.all(np.abs(a - b)[calm] <= tol_abs + tol_rel * np.abs(b)[calm]), (n, gf, float(np.abs(a - b)[calm].max()))
        for j in os_.tolist():
            lo, hi = oro[j], oro[j + 1]
            np.add.at(mass, ((n + od[lo:hi].astype(np.int64)) % D, oport[lo:hi], otgt[lo:hi]), np.abs(ow[lo:hi].astype(np.float64)))
        if diff.size:                                      # divergence on the upswing: re-feed the ring where it exists
            try:
                g.set_state(B.FIELD_RING, o.get_state(oracle_mod.FIELD_RING).astype(np.float32))
            except B.NgError:
                break
    assert n_spk > 50 and len(logged) <= max(3, n_spk // 20), (n_spk, logged)
    g.close()


def test_adex_free_running_rates(oracle_mod, B):
    """Paper-shaped balanced AdEx network at reduced size, 500 ms: population rates agree (C17)."""
    wl = W.balanced_adex(n=5000, k_total=200, n_steps=5000, seed=2)
    o, g = make_adex_pair(wl, oracle_mod, B, debug_input=False)
    assert g.stats().delivery_kernel == 3 and g.stats().step_mode == B.STEP_PERSISTENT
    g.simulate(wl.n_steps); o.simulate(wl.n_steps)
    gs, gi = g.get_spikes(); os_, oi = o.get_spikes()
    t = (wl.n_steps - 1000) * 1e-4
    for first_id, n in wl.pop_ranges():
        rg = np.sum((gi >= first_id) & (gi < first_id + n) & (gs >= 1000)) / n / t
        ro = np.sum((oi >= first_id) & (oi < first_id + n) & (os_ >= 1000)) / n / t
        print(f"adex rates: gpu {rg:.2f} Hz oracle {ro:.2f} Hz")
        assert ro > 1.0 and abs(rg - ro) <= max(0.05 * ro, 0.1), (rg, ro)
    g.close()
