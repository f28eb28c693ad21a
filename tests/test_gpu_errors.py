"""Error behaviour of the C-ABI on a device (include/ng.h states it per entry point): status codes instead of aborts,
messages from ng_last_error, and a simulator that stays usable afterwards."""
import numpy as np
import pytest

from paper_2007_14236_b200 import workloads as W

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    from paper_2007_14236_b200 import binding
    return binding


def code(B, fn, *a, **k):
    with pytest.raises(B.NgError) as e:
        fn(*a, **k)
    return e.value.code


def test_argument_and_state_errors(B):
    g = B.Sim(0.1, 20, 1)
    assert code(B, g.prepare) == B.NG_ERR_STATE                                         # no population
    assert code(B, g.create_population, 0, W.LIF | dict(poisson_rate_hz=0, poisson_weight=0)) == B.NG_ERR_INVALID_ARG
    assert code(B, g.create_population, 10, W.LIF | dict(tau_syn=10.0)) == B.NG_ERR_INVALID_ARG    # tau_m == tau_syn (C19)
    assert code(B, g.create_population, 10, W.LIF | dict(poisson_rate_hz=1e7)) == B.NG_ERR_INVALID_ARG   # Poisson table too short
    first = g.create_population(100, W.LIF | dict(poisson_rate_hz=800.0, poisson_weight=87.8))
    assert first == 0
    assert code(B, g.connect_fixed_indegree, 0, 200, 0, 100, 5, ("const", 1.0), ("const", 1)) == B.NG_ERR_INVALID_ARG   # range
    assert code(B, g.connect_fixed_indegree, 0, 100, 0, 100, 5, ("const", 1.0), ("const", 1), port=2) == B.NG_ERR_INVALID_ARG
    assert code(B, g.get_state, B.FIELD_V) == B.NG_ERR_STATE                            # before prepare
    assert code(B, g.set_option, B.OPT_STEP_MODE, 9) == B.NG_ERR_INVALID_ARG
    g.connect_fixed_indegree(0, 100, 0, 100, 5, ("const", 50.0), ("uniform_int", 1, 20))
    g.prepare()
    assert code(B, g.connect_fixed_indegree, 0, 100, 0, 100, 5, ("const", 1.0), ("const", 1)) == B.NG_ERR_STATE         # after prepare
    assert code(B, g.create_population, 5, W.LIF) == B.NG_ERR_STATE
    assert code(B, g.set_state, B.FIELD_V, np.zeros(101, np.float32)) == B.NG_ERR_INVALID_ARG      # range outside the field
    assert code(B, g.get_state, B.FIELD_LAST_INPUT) == B.NG_ERR_STATE                   # needs NG_DEBUG_INPUT
    assert code(B, g.get_state, B.FIELD_ADEX_W) == B.NG_ERR_STATE                       # no AdEx population
    assert code(B, g.rate_cv) == B.NG_ERR_STATE                                         # statistics not enabled
    g.simulate(50)                                                                      # still usable
    assert g.get_state(B.FIELD_STEP) == 50
    g.close()


def test_delay_beyond_ring_is_overflow(B):
    g = B.Sim(0.1, 8, 1)
    g.create_population(50, W.LIF | dict(poisson_rate_hz=0.0, poisson_weight=0.0))
    g.connect_fixed_indegree(0, 50, 0, 50, 4, ("const", 1.0), ("uniform_int", 1, 9))    # 9 > ring_slots = 8
    assert code(B, g.prepare) == B.NG_ERR_OVERFLOW
    g.close()


def test_spike_record_overflow_keeps_simulating(B):
    wl = W.delivery_microbench(n=2000, K=10, fraction=0.5, n_steps=10, seed=3)
    g = B.Sim(0.1, wl.ring_slots, wl.seed, record_spikes=True, max_recorded_spikes=1500)
    wl.apply(g); g.prepare()
    assert code(B, g.simulate, 5) == B.NG_ERR_OVERFLOW                                 # ~1000 spikes per step
    st = g.stats()
    assert st.steps == 5 and st.spikes > 3000 and st.recorded_dropped > 0
    s, i = g.get_spikes()
    assert s.size == 1500 and np.all(np.diff(s) >= 0)
    g.simulate(2, allow_overflow=True)
    assert g.get_state(B.FIELD_STEP) == 7 and g.stats().events == g.stats().spikes * 10
    g.close()


def test_receptor_port_1_needs_adex_targets(B):
    """Port 1 is the inhibitory conductance of AdEx neurons.  In a LIF-only network the ring has one port, so a port-1
    record would land in the next delay plane (or past the ring); onto LIF targets of a mixed network it would be dropped
    silently.  Both are rejected by ng_prepare."""
    g = B.Sim(0.1, 20, 1)
    g.create_population(100, W.LIF | dict(poisson_rate_hz=800.0, poisson_weight=87.8))
    g.connect_fixed_indegree(0, 100, 0, 100, 5, ("const", 1.0), ("uniform_int", 1, 20), port=1)
    assert code(B, g.prepare) == B.NG_ERR_INVALID_ARG
    g.close()
    ax = dict(W.ADEX); ax.update(poisson_rate_hz=20000.0, poisson_weight=0.37)
    g = B.Sim(0.1, 20, 1)
    g.create_population(100, W.LIF | dict(poisson_rate_hz=800.0, poisson_weight=87.8))
    g.create_population(100, ax)
    g.connect_fixed_indegree(0, 200, 50, 150, 5, ("const", 0.35), ("uniform_int", 1, 20), port=1)     # targets 50..199: half LIF
    assert code(B, g.prepare) == B.NG_ERR_INVALID_ARG
    g.close()
    g = B.Sim(0.1, 20, 1)
    g.create_population(100, W.LIF | dict(poisson_rate_hz=800.0, poisson_weight=87.8))
    g.create_population(100, ax)
    g.connect_fixed_indegree(0, 200, 100, 100, 5, ("const", 0.35), ("uniform_int", 1, 20), port=1)    # AdEx targets only
    g.connect_fixed_indegree(0, 200, 0, 100, 5, ("const", 50.0), ("uniform_int", 1, 20))
    g.prepare()
    g.simulate(30)
    assert g.get_state(B.FIELD_STEP) == 30
    g.close()


def test_trace_option_can_be_switched_off_and_on(B):
    wl = W.brunel_tiny(n_steps=50)
    g = B.Sim(0.1, wl.ring_slots, wl.seed)
    wl.apply(g); g.prepare()
    before = None
    for k in range(3):
        g.set_option(B.OPT_TRACE, 1)
        if before is None:
            before = len(g._tensors)
        assert len(g._tensors) == before               # the saved buffer is reused, nothing new is allocated
        g.simulate(10)
        assert g.trace().shape[0] == 64
        g.set_option(B.OPT_TRACE, 0)
        g.simulate(10)
    g.close()


def test_pipelined_window_backend_rules(B):
    """Delivery kernel 6 exists as a persistent cooperative kernel with a neuron update: not in delivery-only mode, not
    with ring_slots = 1, not sharded, and — like kernels 4 and 5 — only when chosen before ng_prepare."""
    wl = W.delivery_microbench(n=5000, K=50, fraction=0.05, n_steps=10, seed=2)
    g = B.Sim(0.1, wl.ring_slots, wl.seed)
    wl.apply(g); g.set_option(B.OPT_DELIVERY_KERNEL, 6)
    assert code(B, g.prepare) == B.NG_ERR_INVALID_ARG                                   # delivery-only mode
    g.close()
    g = B.Sim(0.1, 1, 1)
    g.create_population(100, W.LIF | dict(poisson_rate_hz=800.0, poisson_weight=87.8))
    g.connect_fixed_indegree(0, 100, 0, 100, 5, ("const", 50.0), ("const", 1))
    g.set_option(B.OPT_DELIVERY_KERNEL, 6)
    assert code(B, g.prepare) == B.NG_ERR_INVALID_ARG                                   # one ring slot: no delay >= 2 exists
    g.close()
    g = B.Sim(0.1, 20, 1, rank=0, world=2)
    assert code(B, g.set_option, B.OPT_DELIVERY_KERNEL, 6) == B.NG_ERR_INVALID_ARG      # one GPU only
    g.close()
    wl = W.brunel_tiny(n_steps=50)
    g = B.Sim(0.1, wl.ring_slots, wl.seed)
    wl.apply(g); g.prepare()
    assert code(B, g.set_option, B.OPT_DELIVERY_KERNEL, 6) == B.NG_ERR_STATE            # after ng_prepare
    g.close()
    g = B.Sim(0.1, wl.ring_slots, wl.seed)
    wl.apply(g); g.set_option(B.OPT_DELIVERY_KERNEL, 6); g.prepare()
    g.set_option(B.OPT_STEP_MODE, 0)                                                    # ignored: kernel 6 is persistent only
    g.set_state(B.FIELD_V, wl.initial_v())
    g.simulate(50)
    st = g.stats()
    assert st.delivery_kernel == 6 and st.step_mode == B.STEP_PERSISTENT and st.spikes > 150
    assert code(B, g.set_state, B.FIELD_RING, np.zeros(1000 * 20, np.float32)) == B.NG_ERR_STATE   # two planes: read-only
    assert g.get_state(B.FIELD_RING).size == 1000 * 20
    g.close()
