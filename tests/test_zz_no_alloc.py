"""ng_deliver_noalloc (include/ng.h, csrc/ng_noalloc.cu): spike delivery with its ring in a static device array, for
callers that cannot call cudaMalloc.  Checked against the EXISTING path — an ng_sim in delivery-only mode (reading C8)
with delivery kernel 1 — on the same connection arrays and the same spikes, two sequences in a row (the static ring
keeps the last call's contents; the second sequence, another network, starts with reset):

  * per step, input_out (the plane the step consumes) against NG_FIELD_LAST_INPUT of the existing path;
  * after the last step, the remaining ring contents (drained by ring_slots more calls without spikes) against
    NG_FIELD_RING of the existing path.

Both sides add the same fp32 weights to the same cells with red.global.add.f32 in an order the hardware chooses: the
tolerance is the one tests/test_gpu_delivery.py uses, 1e-5 of the L1 mass of the cell (C12), and cells are
non-zero on one side exactly where they are on the other.

The file sorts last on purpose: the run uses pytest -x.  It must pass alone in a fresh process and after
the other tests (it makes no assumption about what the static array holds when it starts)."""
import numpy as np
import pytest

from paper_2007_14236_b200 import workloads as W

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    from paper_2007_14236_b200 import binding
    return binding


def existing_path(B, wl, steps):
    """The existing delivery path one step at a time: per-step consumed planes, spike ids per step, the final ring, and the
    connection arrays copied into device tensors."""
    import torch
    g = B.Sim(0.1, wl.ring_slots, wl.seed, record_spikes=True, max_recorded_spikes=1 << 22, debug_input=True)
    wl.apply(g); g.prepare()
    g.set_option(B.OPT_DELIVERY_KERNEL, 1)
    g.set_option(B.OPT_STEP_MODE, B.STEP_LAUNCH)
    N = wl.n_neurons
    consumed, spikes = [], []
    for n in range(steps):
        g.simulate(1)
        consumed.append(g.get_state(B.FIELD_LAST_INPUT).astype(np.float64))
        s, i = g.get_spikes()
        assert np.all(s == n)
        spikes.append(np.sort(i).astype(np.int32))
    ring = g.get_state(B.FIELD_RING).astype(np.float64).reshape(wl.ring_slots, N)
    ro_h = g.row_offsets(); tgt_h, w_h, d_h = g.records()
    dev = torch.device("cuda:0")
    ro = torch.from_numpy(ro_h).to(dev); tgt = torch.from_numpy(tgt_h).to(dev)
    w = torch.from_numpy(w_h).to(dev); d = torch.from_numpy(d_h).to(dev)
    g.close()
    return consumed, spikes, ring, (ro_h, tgt_h, w_h, d_h), (ro, tgt, w, d)


def l1_mass(host_csr, spikes, N, D, upto):
    """|w| delivered to every ring cell by the spikes of steps < upto and not consumed before step upto; plus, per step
    n < upto, the mass of the plane step n consumed."""
    ro, tgt, w, d = host_csr
    mass = np.zeros((D, N))
    consumed = []
    for n in range(upto):
        consumed.append(mass[n % D].copy())
        mass[n % D] = 0.0
        for j in spikes[n]:
            lo, hi = ro[j], ro[j + 1]
            keep = tgt[lo:hi] >= 0
            np.add.at(mass, ((n + d[lo:hi][keep].astype(np.int64)) % D, tgt[lo:hi][keep]), np.abs(w[lo:hi][keep]).astype(np.float64))
    return mass, consumed


def run_sequence(B, wl, steps):
    import torch
    consumed, spikes, ring, host_csr, (ro, tgt, w, d) = existing_path(B, wl, steps)
    N, D = wl.n_neurons, wl.ring_slots
    assert N * D <= B.NOALLOC_MAX_CELLS and sum(s.size for s in spikes) > 0
    mass, cmass = l1_mass(host_csr, spikes, N, D, steps)
    dev = torch.device("cuda:0")
    out = torch.empty(N, dtype=torch.float32, device=dev)
    stream = torch.cuda.current_stream().cuda_stream
    touched = 0
    for n in range(steps):
        ids = torch.from_numpy(spikes[n]).to(dev)
        B.deliver_noalloc(ro, tgt, w, d, ids, ids.numel(), N, D, n, out, reset=(n == 0), stream=stream)
        got = out.cpu().numpy().astype(np.float64)
        assert np.array_equal(got != 0, consumed[n] != 0), n
        assert np.all(np.abs(got - consumed[n]) <= 1e-5 * cmass[n] + 1e-12), (n, float(np.abs(got - consumed[n]).max()))
        touched += np.count_nonzero(got)
    assert touched > 0
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]                      # no torch kernel or device allocation until the check
    for k in range(D):                                        # drain: what is still in flight after the last step
        n = steps + k
        B.deliver_noalloc(ro, tgt, w, d, None, 0, N, D, n, out, stream=stream)
        got = out.cpu().numpy().astype(np.float64)
        want = ring[n % D]
        assert np.array_equal(got != 0, want != 0), n
        assert np.all(np.abs(got - want) <= 1e-5 * mass[n % D] + 1e-12), (n, float(np.abs(got - want).max()))
    assert B.deliver_noalloc_check(stream) == 0
    assert torch.cuda.mem_get_info()[0] == free0              # the D + 1 calls above allocated nothing on the device
    assert np.count_nonzero(ring) > 0
    B.deliver_noalloc(ro, tgt, w, d, None, 0, N, D, steps + D, out, stream=stream)      # everything consumed: the ring is empty
    assert not out.any().item()


def test_no_alloc_delivery_matches_existing_path_twice(B):
    """Two sequences in a row on the shared static ring: K = 100 (rows of 25 vectors), then K = 37 (rows with padding
    records) on a smaller network with another ring length, the second one started on a ring the first one has used."""
    run_sequence(B, W.delivery_microbench(n=20000, K=100, fraction=0.05, n_steps=70, seed=5), 70)    # 70 > D = 64: the ring wraps
    run_sequence(B, W.delivery_microbench(n=15000, K=37, fraction=0.03, n_steps=70, seed=6), 70)


def test_no_alloc_without_reset_keeps_last_contents(B):
    """The array keeps the last call's contents: a spike delivered in one call arrives in a later call."""
    import torch
    dev = torch.device("cuda:0")
    N, D = 1000, 8
    ro = torch.tensor([0, 4, 8], dtype=torch.int64, device=dev)
    tgt = torch.tensor([5, 6, 999, -1, 5, 7, -1, -1], dtype=torch.int32, device=dev)
    w = torch.tensor([1.5, -2.0, 0.25, 9.0, 4.0, 8.0, 9.0, 9.0], dtype=torch.float32, device=dev)
    d = torch.tensor([1, 3, 8, 1, 3, 3, 1, 1], dtype=torch.uint8, device=dev)
    out = torch.empty(N, dtype=torch.float32, device=dev)
    ids = torch.tensor([0, 1], dtype=torch.int32, device=dev)
    B.deliver_noalloc(ro, tgt, w, d, ids, 2, N, D, 10, out, reset=True)
    assert not out.any().item()
    want = {11: {5: 1.5}, 13: {6: -2.0, 5: 4.0, 7: 8.0}, 18: {999: 0.25}}
    for n in range(11, 20):
        B.deliver_noalloc(ro, tgt, w, d, None, 0, N, D, n, out)
        got = out.cpu().numpy()
        exp = np.zeros(N, np.float32)
        for i, v in want.get(n, {}).items():
            exp[i] = v
        assert np.array_equal(got, exp), n
    assert B.deliver_noalloc_check() == 0


def test_no_alloc_rejects_sizes_beyond_the_static_array(B):
    import torch
    out = torch.empty(16, dtype=torch.float32, device="cuda:0")
    with pytest.raises(B.NgError) as e:
        B.deliver_noalloc(None, None, None, None, None, 0, (B.NOALLOC_MAX_CELLS // 64) + 1, 64, 0, out)
    assert e.value.code == B.NG_ERR_INVALID_ARG and "NG_NOALLOC_MAX_CELLS" in str(e.value)
    with pytest.raises(B.NgError):
        B.deliver_noalloc(None, None, None, None, None, 0, 16, 0, 0, out)
    with pytest.raises(B.NgError):
        B.deliver_noalloc(None, None, None, None, None, 3, 16, 4, 0, out)          # spikes without arrays
    # out-of-range records are skipped and reported by the check
    dev = torch.device("cuda:0")
    ro = torch.tensor([0, 4], dtype=torch.int64, device=dev)
    tgt = torch.tensor([1, 16, 2, 3], dtype=torch.int32, device=dev)
    w = torch.ones(4, dtype=torch.float32, device=dev)
    d = torch.tensor([1, 1, 5, 0], dtype=torch.uint8, device=dev)
    ids = torch.tensor([0, 7], dtype=torch.int32, device=dev)
    B.deliver_noalloc(ro, tgt, w, d, ids, 2, 16, 4, 0, out, reset=True)
    with pytest.raises(B.NgError) as e:
        B.deliver_noalloc_check()
    assert e.value.code == B.NG_ERR_OVERFLOW
    assert B.deliver_noalloc_check() == 0                      # the count was cleared
    B.deliver_noalloc(ro, tgt, w, d, None, 0, 16, 4, 1, out)
    got = out.cpu().numpy()
    assert got[1] == 1.0 and np.count_nonzero(got) == 1
