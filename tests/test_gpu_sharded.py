"""Target-sharded multi-GPU path on ONE GPU: the `world` shards of a network
run as handles of one process on one stream, stepped half by half (binding.ShardGroup / ng_shard_phase), so the per-step
spike exchange — peer stores into the other shards' receive buffers, step-stamped flags, gather into the local spike
array — is exactly the code that runs across GPUs, while no kernel ever waits for another (B200_PROFILING.md).

Bars: every shard stores exactly the oracle's connections whose target it owns (bit-exact, local target indices); the
union of the shards' dynamics equals the oracle in lockstep and the one-GPU run spike for spike; delivery-only rings
equal the oracle's for every delivery backend that runs sharded (1, 2, 4, 5)."""
import numpy as np
import pytest

from paper_2007_14236_b200 import workloads as W

from helpers import Shadow

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    from paper_2007_14236_b200 import binding
    return binding


def make_group(B, wl, world, pre_options=None, **kw):
    g = B.ShardGroup(world, 0.1, wl.ring_slots, wl.seed, **kw)
    wl.apply(g)
    for opt, val in (pre_options or {}).items():
        g.set_option(opt, val)
    g.prepare()
    return g


@pytest.mark.parametrize("world", [2, 3])
def test_shards_hold_the_oracle_structure_restricted_to_their_targets(oracle_mod, B, world):
    wl = W.microcircuit(scale_div=20, n_steps=10, indegree_div=2)
    o = oracle_mod.Oracle(0.1, wl.ring_slots, wl.seed); wl.apply(o); o.prepare()
    g = make_group(B, wl, world)
    N = wl.n_neurons
    assert [r for r in g.ranges] == [B.shard_range(N, r, world) for r in range(world)]
    assert sum(n for _, n in g.ranges) == N and g.ranges[0][0] == 0
    osrc, otgt, ow, od, oro = o.get_connections()
    total = 0
    for sh, (f0, nloc) in zip(g.shards, g.ranges):
        st = sh.stats()
        assert (st.shard_rank, st.shard_world, st.id_first, st.n_neurons, st.n_sources) == (sh.rank, world, f0, nloc, N)
        ro = sh.row_offsets(); tgt, w, d = sh.records(); go = sh.group_offsets().astype(np.int64)
        src = np.repeat(np.arange(N, dtype=np.int32), np.diff(ro))
        keep = tgt >= 0
        assert tgt[keep].max() < nloc                       # local target indices (one receptor port)
        mine = (otgt >= f0) & (otgt < f0 + nloc)
        assert keep.sum() == mine.sum() == st.n_connections
        total += int(keep.sum())
        a = np.lexsort((w[keep].view(np.uint32), tgt[keep], d[keep], src[keep]))
        b = np.lexsort((ow[mine].view(np.uint32), otgt[mine], od[mine], osrc[mine]))
        assert np.array_equal(src[keep][a], osrc[mine][b]) and np.array_equal(tgt[keep][a] + f0, otgt[mine][b])
        assert np.array_equal(d[keep][a], od[mine][b])
        assert np.all(np.abs(w[keep][a].view(np.uint32).astype(np.int64) - ow[mine][b].view(np.uint32).astype(np.int64)) <= 1)
        # rows padded to 4, groups = prefix sums of the per-(source, delay) histogram of the shard's records
        hist = np.zeros((N, wl.ring_slots + 1), np.int64)
        np.add.at(hist, (osrc[mine], od[mine].astype(np.int64)), 1)
        assert np.array_equal(go, np.cumsum(hist, axis=1)) and np.array_equal(np.diff(ro), (go[:, -1] + 3) // 4 * 4)
    assert total == o.n_connections
    g.close()


@pytest.mark.parametrize("world,kernel", [(2, 1), (3, 1), (2, 2), (2, 4), (2, 5)])
def test_sharded_lockstep_against_the_oracle(oracle_mod, B, world, kernel):
    """The oracle's state (fp32-rounded) is fed to the shards every step; spike lists must be identical except within 1e-4 mV
    of threshold, consumed inputs within 1e-5 of their L1 mass (C12), V within 1e-4 mV — the one-GPU bars."""
    wl = W.microcircuit(scale_div=40, n_steps=150, indegree_div=8)
    o = oracle_mod.Oracle(0.1, wl.ring_slots, wl.seed); wl.apply(o); o.prepare()
    g = make_group(B, wl, world, pre_options={B.OPT_DELIVERY_KERNEL: kernel}, debug_input=True)
    assert all(st.delivery_kernel == kernel and st.step_mode != B.STEP_PERSISTENT for st in g.stats())
    v0 = wl.initial_v()
    o.set_state(oracle_mod.FIELD_V, v0.astype(np.float64)); g.set_state(B.FIELD_V, v0)
    N, D = wl.n_neurons, wl.ring_slots
    sh = Shadow(o, wl, oracle_mod)
    n_spk, log = 0, []
    for n in range(150):
        V = o.get_state(oracle_mod.FIELD_V); I = o.get_state(oracle_mod.FIELD_I_SYN); R = o.get_state(oracle_mod.FIELD_REFR)
        V32, I32 = V.astype(np.float32), I.astype(np.float32)
        g.set_state(B.FIELD_V, V32); g.set_state(B.FIELD_I_SYN, I32); g.set_state(B.FIELD_REFR, R)
        in_or = o.get_state(oracle_mod.FIELD_RING, N, first=(n % D) * N)
        abs_in = sh.consume(n)
        v_pre = np.where(R == 0, sh.E_L + sh.P22 * (V32.astype(np.float64) - sh.E_L) + sh.P21 * I32.astype(np.float64), -1e9)
        near = np.abs(v_pre - sh.V_th) < 1e-4
        g.simulate(1); o.simulate(1, record=False)
        gs = g.last_spikes(); os_ = np.sort(o.last_spikes())
        diff = np.setxor1d(gs, os_)
        assert np.all(near[diff]), (n, diff[~near[diff]][:10])
        n_spk += os_.size
        gin = g.get_state(B.FIELD_LAST_INPUT).astype(np.float64)
        assert np.all(np.abs(gin - in_or) <= 1e-5 * abs_in + 1e-12), (n, float(np.abs(gin - in_or).max()))
        keep = np.ones(N, bool); keep[diff] = False
        gV = g.get_state(B.FIELD_V).astype(np.float64)
        assert np.all(np.abs(gV - o.get_state(oracle_mod.FIELD_V))[keep] <= 1e-4)
        assert np.array_equal(g.get_state(B.FIELD_REFR)[keep], o.get_state(oracle_mod.FIELD_REFR)[keep])
        sh.deliver(n, os_)
        if diff.size:
            log.append((n, diff.tolist()))
            break                                            # the shards' pending inputs cannot be re-fed
    assert n_spk > 60 and len(log) <= 1, (n_spk, log)
    g.close()


@pytest.mark.parametrize("world", [2, 4])
def test_sharded_free_run_equals_one_gpu_cfg1(oracle_mod, B, world):
    """BASELINE.json configs[1] (7,718 neurons, 29.9e6 connections): the union of the shards' spikes equals the one-GPU run
    and the oracle spike for spike over the first steps, and every shard's spike record is the whole network's."""
    wl = W.microcircuit(10, 400)
    v0 = wl.initial_v()
    g = make_group(B, wl, world, max_recorded_spikes=1 << 22)
    g.set_state(B.FIELD_V, v0)
    assert sum(st.n_connections for st in g.stats()) == 29_892_043
    one = B.Sim(0.1, wl.ring_slots, wl.seed, record_spikes=True)
    wl.apply(one); one.prepare(); one.set_state(B.FIELD_V, v0)
    o = oracle_mod.Oracle(0.1, wl.ring_slots, wl.seed); wl.apply(o); o.prepare()
    o.set_state(oracle_mod.FIELD_V, v0.astype(np.float64))
    steps = 400
    g.simulate(steps); one.simulate(steps); o.simulate(steps)
    gs, gi = g.get_spikes(); s1, i1 = one.get_spikes(); os_, oi = o.get_spikes()
    first = 60                                               # before fp32 summation order / fp64 can separate the runs
    a = set(zip(gs[gs < first].tolist(), gi[gs < first].tolist()))
    b = set(zip(s1[s1 < first].tolist(), i1[s1 < first].tolist()))
    c = set(zip(os_[os_ < first].tolist(), oi[os_ < first].tolist()))
    assert len(c) > 1500 and len(a ^ c) <= 2 and len(a ^ b) <= 2, (len(a), len(b), len(c), sorted(a ^ c)[:5])
    # afterwards the trajectories may separate: population rates over the whole run agree (C17; 40 ms is short: 10 %)
    for first_id, n in wl.pop_ranges():
        rg = np.sum((gi >= first_id) & (gi < first_id + n)) / n; r1 = np.sum((i1 >= first_id) & (i1 < first_id + n)) / n
        assert abs(rg - r1) <= max(0.1 * r1, 0.02), (rg, r1)
    assert sum(st.events for st in g.stats()) == pytest.approx(one.stats().events, rel=0.02)
    assert all(st.spikes == gs.size for st in g.stats())
    g.close(); one.close()


@pytest.mark.parametrize("kernel,world", [(1, 2), (2, 3), (4, 2), (5, 2), (5, 4)])
def test_sharded_delivery_only_matches_oracle(oracle_mod, B, kernel, world):
    """Delivery alone (reading C8), fixed out-degree — every source has targets on every shard: injected spikes bit-exact
    (each shard injects for the sources it owns, Philox keyed by the global id), ring contents equal to the oracle's."""
    n, steps, K = 20000, 70, 200
    wl = W.delivery_microbench(n=n, K=K, fraction=0.02, n_steps=steps, seed=5)
    o = oracle_mod.Oracle(0.1, wl.ring_slots, wl.seed); wl.apply(o); o.prepare()
    g = make_group(B, wl, world, pre_options={B.OPT_DELIVERY_KERNEL: kernel})
    g.simulate(steps); o.simulate(steps)
    gs, gi = g.get_spikes(); os_, oi = o.get_spikes()
    ko = np.lexsort((oi, os_))
    assert np.array_equal(gs, os_[ko]) and np.array_equal(gi, oi[ko]) and gs.size > 20000
    assert sum(st.events for st in g.stats()) == o.n_events == gs.size * K
    gr = g.get_state(B.FIELD_RING).astype(np.float64)
    orr = o.get_state(oracle_mod.FIELD_RING)
    assert np.count_nonzero(orr) > 0 and np.array_equal(gr != 0, orr != 0)
    assert np.all(np.abs(gr - orr) <= 1e-4 * np.abs(orr) + 1e-9), float(np.abs(gr - orr).max())
    g.close()


def test_sharded_adex_two_ports(oracle_mod, B):
    """AdEx network with two receptor ports in two shards: same spikes as the oracle over the first steps, free-running."""
    wl = W.balanced_adex(n=3000, k_total=100, n_steps=400, seed=3)
    v0 = wl.initial_v()
    g = make_group(B, wl, 2)
    g.set_state(B.FIELD_V, v0)
    o = oracle_mod.Oracle(0.1, wl.ring_slots, wl.seed); wl.apply(o); o.prepare()
    o.set_state(oracle_mod.FIELD_V, v0.astype(np.float64))
    g.simulate(400); o.simulate(400)
    gs, gi = g.get_spikes(); os_, oi = o.get_spikes()
    first = 200
    a = set(zip(gs[gs < first].tolist(), gi[gs < first].tolist())); c = set(zip(os_[os_ < first].tolist(), oi[os_ < first].tolist()))
    assert len(c) > 100 and len(a ^ c) <= max(2, len(c) // 100), (len(a), len(c))
    assert abs(gs.size - os_.size) <= 0.1 * os_.size
    g.close()


def test_sharded_api_rules(B):
    wl = W.brunel_tiny(n_steps=10)
    g = B.Sim(0.1, wl.ring_slots, wl.seed, rank=1, world=2)
    wl.apply(g)
    with pytest.raises(B.NgError):
        g.set_option(B.OPT_DELIVERY_KERNEL, 3)               # pipelined kernel: one GPU only
    g.prepare()
    st = g.stats()
    assert (st.id_first, st.n_neurons, st.n_sources) == (500, 500, 1000)
    with pytest.raises(B.NgError):
        g.simulate(1)                                        # peers not attached
    with pytest.raises(B.NgError):
        g.enable_statistics()
    h, p = g.exchange_handle()
    assert len(h) == 64 and p
    with pytest.raises(B.NgError):
        g.exchange_attach(1, ptr=p)                          # own rank
    g.close()
    with pytest.raises(B.NgError):
        B.Sim(0.1, 20, 1, rank=2, world=2)
