"""Thin ctypes binding of libng.so (include/ng.h).  Argument marshalling only: every step of the hot path runs in
the CUDA kernels behind the C-ABI.  PyTorch supplies device memory (allocator callbacks) and the CUDA stream.

There is no CPU fallback: importing this module loads libng.so and raises if it is missing or cannot be built.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import build as _build

NG_OK, NG_ERR_INVALID_ARG, NG_ERR_STATE, NG_ERR_OOM, NG_ERR_CUDA, NG_ERR_OVERFLOW = 0, -1, -2, -3, -4, -5
NG_RECORD_SPIKES, NG_DEBUG_INPUT = 1, 2
FIELD_V, FIELD_I_SYN, FIELD_REFR, FIELD_RING, FIELD_STEP, FIELD_LAST_INPUT = 0, 1, 2, 3, 4, 5
FIELD_ADEX_W, FIELD_ADEX_G_EX, FIELD_ADEX_Y_EX, FIELD_ADEX_G_IN, FIELD_ADEX_Y_IN, FIELD_ADEX_H = 6, 7, 8, 9, 10, 11
DIST_CONST, DIST_NORMAL_CLIPPED, DIST_UNIFORM_INT = 0, 1, 2
(OPT_STEP_MODE, OPT_STEPS_PER_GRAPH, OPT_DELIVERY_KERNEL, OPT_DELIVER_BLOCKS, OPT_PROFILE, OPT_ASYNC,
 OPT_SORT_SEGMENTS, OPT_PREFETCH, OPT_TRACE, OPT_PERSISTENT_THREADS, OPT_QUEUE_CAPACITY) = range(11)
STEP_GRAPH, STEP_LAUNCH, STEP_PERSISTENT, STEP_AUTO = 0, 1, 2, 3

EXPORTS = ["ng_create", "ng_destroy", "ng_last_error", "ng_create_population", "ng_connect_fixed_indegree",
           "ng_connect_fixed_outdegree", "ng_set_bypass", "ng_set_option", "ng_prepare", "ng_set_state",
           "ng_get_state", "ng_simulate", "ng_get_spikes", "ng_get_last_spikes", "ng_copy_row_offsets",
           "ng_copy_group_offsets", "ng_copy_records", "ng_get_connections", "ng_get_stats", "ng_get_trace", "ng_probe",
           "ng_create_population_adex", "ng_connect_fixed_indegree_port", "ng_connect_fixed_outdegree_port",
           "ng_enable_statistics", "ng_get_rate_cv", "ng_get_correlations",
           "ng_shard_range", "ng_set_shard", "ng_exchange_handle", "ng_exchange_attach", "ng_shard_phase",
           "ng_deliver_noalloc", "ng_deliver_noalloc_check", "ng_noalloc_last_error"]
NOALLOC_MAX_CELLS = 1 << 22


class NgConfig(C.Structure):
    _fields_ = [("dt_ms", C.c_double), ("ring_slots", C.c_int32), ("flags", C.c_uint32), ("seed", C.c_uint64),
                ("max_recorded_spikes", C.c_int64), ("device", C.c_int32), ("reserved", C.c_int32)]


_ALLOC_FN = C.CFUNCTYPE(C.c_void_p, C.c_size_t, C.c_void_p)
_FREE_FN = C.CFUNCTYPE(None, C.c_void_p, C.c_void_p)


class NgAllocator(C.Structure):
    _fields_ = [("alloc", _ALLOC_FN), ("free", _FREE_FN), ("user", C.c_void_p)]


class NgLifParams(C.Structure):
    _fields_ = [(k, C.c_double) for k in
                ("C_m", "tau_m", "tau_syn", "E_L", "V_th", "V_reset", "t_ref_ms", "I_e",
                 "poisson_rate_hz", "poisson_weight")]


_ADEX_SCALARS = ("C_m", "g_L", "E_L", "V_T", "Delta_T", "tau_w", "a", "b", "V_reset", "V_peak", "E_ex", "E_in", "tau_syn",
                 "I_e", "poisson_rate_hz", "poisson_weight")


class NgAdexParams(C.Structure):
    _fields_ = [(k, C.c_double) for k in _ADEX_SCALARS] + [("tol", C.c_double * 6), ("h_min", C.c_double)]


def _adex(params: dict) -> NgAdexParams:
    p = NgAdexParams(**{k: float(params.get(k, 0.0)) for k in _ADEX_SCALARS})
    for i, t in enumerate(params["tol"]):
        p.tol[i] = float(t)
    p.h_min = float(params["h_min"])
    return p


class NgDist(C.Structure):
    _fields_ = [("kind", C.c_int32), ("pad", C.c_int32), ("a", C.c_double), ("b", C.c_double),
                ("lo", C.c_double), ("hi", C.c_double)]


class NgStats(C.Structure):
    _fields_ = [("steps", C.c_uint64), ("spikes", C.c_uint64), ("events", C.c_uint64),
                ("recorded_dropped", C.c_uint64), ("n_neurons", C.c_int64), ("n_connections", C.c_int64),
                ("n_records_padded", C.c_int64), ("max_row_records", C.c_int64), ("build_ms", C.c_double),
                ("ms_update", C.c_double), ("ms_deliver", C.c_double), ("launches_update", C.c_uint64),
                ("launches_deliver", C.c_uint64), ("launches_other", C.c_uint64), ("delivery_kernel", C.c_int32),
                ("step_mode", C.c_int32), ("n_sources", C.c_int64), ("shard_rank", C.c_int32), ("shard_world", C.c_int32),
                ("id_first", C.c_int32), ("step_kernel", C.c_int32)]


class NgError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"ng error {code}: {msg}")
        self.code = code


_lib = None


def load_library(path: str | None = None):
    """Load libng.so (building it with nvcc if it is missing or stale).  Raises on failure — no fallback."""
    global _lib
    if _lib is not None and path is None:
        return _lib
    p = path or _build.build_lib()
    if not os.path.exists(p):
        raise ImportError(f"libng.so not found at {p}; run `python -m paper_2007_14236_b200.build`")
    L = C.CDLL(p)
    vp, i32, i64 = C.c_void_p, C.c_int32, C.c_int64
    L.ng_create.argtypes = [C.POINTER(NgConfig), C.POINTER(NgAllocator), vp, C.POINTER(vp)]
    L.ng_destroy.argtypes = [vp]
    L.ng_last_error.argtypes = [vp]
    L.ng_last_error.restype = C.c_char_p
    L.ng_create_population.argtypes = [vp, i32, C.POINTER(NgLifParams), C.POINTER(i32)]
    for fn in (L.ng_connect_fixed_indegree, L.ng_connect_fixed_outdegree):
        fn.argtypes = [vp, i32, i32, i32, i32, i32, C.POINTER(NgDist), C.POINTER(NgDist)]
    for fn in (L.ng_connect_fixed_indegree_port, L.ng_connect_fixed_outdegree_port):
        fn.argtypes = [vp, i32, i32, i32, i32, i32, C.POINTER(NgDist), C.POINTER(NgDist), i32]
    L.ng_create_population_adex.argtypes = [vp, i32, C.POINTER(NgAdexParams), C.POINTER(i32)]
    L.ng_set_bypass.argtypes = [vp, i32, C.c_double]
    L.ng_set_option.argtypes = [vp, i32, i64]
    L.ng_prepare.argtypes = [vp]
    L.ng_set_state.argtypes = [vp, i32, vp, i64, i64]
    L.ng_get_state.argtypes = [vp, i32, vp, i64, i64]
    L.ng_simulate.argtypes = [vp, i64]
    L.ng_get_spikes.argtypes = [vp, vp, vp, i64, C.POINTER(i64)]
    L.ng_get_last_spikes.argtypes = [vp, vp, i64, C.POINTER(i64)]
    L.ng_copy_row_offsets.argtypes = [vp, vp]
    L.ng_copy_group_offsets.argtypes = [vp, vp]
    L.ng_copy_records.argtypes = [vp, i64, i64, vp, vp, vp]
    L.ng_get_connections.argtypes = [vp, i32, vp, vp, vp, i64, C.POINTER(i64)]
    L.ng_get_stats.argtypes = [vp, C.POINTER(NgStats)]
    L.ng_get_trace.argtypes = [vp, vp, i64, C.POINTER(i64), C.POINTER(i32)]
    L.ng_enable_statistics.argtypes = [vp, i64, i32, i32, i32]
    L.ng_get_rate_cv.argtypes = [vp, vp, vp, i64]
    L.ng_get_correlations.argtypes = [vp, i32, vp, i64, C.POINTER(i32), C.POINTER(i32)]
    L.ng_probe.argtypes = [i32, i32, i64, C.POINTER(C.c_double)]
    L.ng_shard_range.argtypes = [i32, i32, i32, C.POINTER(i32), C.POINTER(i32)]
    L.ng_set_shard.argtypes = [vp, i32, i32]
    L.ng_exchange_handle.argtypes = [vp, vp, C.POINTER(vp)]
    L.ng_exchange_attach.argtypes = [vp, i32, vp, vp]
    L.ng_shard_phase.argtypes = [vp, i32]
    L.ng_deliver_noalloc.argtypes = [vp, vp, vp, vp, vp, i32, vp, i32, i32, i32, i64, i32, vp]
    L.ng_deliver_noalloc_check.argtypes = [vp, C.POINTER(i64)]
    L.ng_noalloc_last_error.argtypes = []
    L.ng_noalloc_last_error.restype = C.c_char_p
    for name in EXPORTS:
        if name not in ("ng_last_error", "ng_noalloc_last_error"):
            getattr(L, name).restype = i32
    if path is None:
        _lib = L
    return L


def probe(kind: int, footprint_bytes: int = 4 << 20, device: int = 0) -> float:
    """ng_probe: kind 0 stream bytes/s, 1 scattered reductions/s, 2 streamed records + reductions events/s."""
    out = C.c_double()
    rc = load_library().ng_probe(device, kind, footprint_bytes, C.byref(out))
    if rc != NG_OK:
        raise NgError(rc, "ng_probe failed")
    return out.value


def _dev_ptr(t):
    return 0 if t is None else t.data_ptr()


def deliver_noalloc(row_offsets, tgt, w, delay, spike_ids, n_spikes: int, n_targets: int, ring_slots: int, step: int,
                    input_out, reset: bool = False, stream: int = 0) -> None:
    """ng_deliver_noalloc: one delivery step on caller-owned DEVICE tensors (int64 row offsets, int32 targets, float32
    weights, uint8 delays, int32 spike ids, float32 output), the ring in the library's static 16 MiB device array.
    Enqueues on `stream` (a raw cudaStream_t, 0 = default) of the current device and returns; allocates nothing."""
    L = load_library()
    rc = L.ng_deliver_noalloc(stream, _dev_ptr(row_offsets), _dev_ptr(tgt), _dev_ptr(w), _dev_ptr(delay),
                              0 if row_offsets is None else row_offsets.numel() - 1, _dev_ptr(spike_ids), n_spikes,
                              n_targets, ring_slots, step, int(bool(reset)), _dev_ptr(input_out))
    if rc != NG_OK:
        raise NgError(rc, L.ng_noalloc_last_error().decode())


def deliver_noalloc_check(stream: int = 0) -> int:
    """ng_deliver_noalloc_check: synchronises; raises if records or spike ids were skipped as out of range since the last check."""
    L = load_library()
    bad = C.c_int64()
    rc = L.ng_deliver_noalloc_check(stream, C.byref(bad))
    if rc != NG_OK:
        raise NgError(rc, L.ng_noalloc_last_error().decode())
    return bad.value


def _lif(params: dict) -> NgLifParams:
    return NgLifParams(**{k: float(params.get(k, 0.0)) for k, _ in NgLifParams._fields_})


def _dist(d) -> NgDist:
    """d = ("const", a) | ("normal", mean, sd[, lo, hi]) | ("uniform_int", lo, hi)."""
    kind = d[0]
    if kind == "const":
        return NgDist(DIST_CONST, 0, float(d[1]), 0.0, 0.0, 0.0)
    if kind == "normal":
        lo = float(d[3]) if len(d) > 3 else -np.inf
        hi = float(d[4]) if len(d) > 4 else np.inf
        return NgDist(DIST_NORMAL_CLIPPED, 0, float(d[1]), float(d[2]), lo, hi)
    if kind == "uniform_int":
        return NgDist(DIST_UNIFORM_INT, 0, 0.0, 0.0, float(d[1]), float(d[2]))
    raise ValueError(kind)


def _ptr(x):
    """Host numpy array or torch tensor (host or device) -> raw address."""
    if isinstance(x, np.ndarray):
        assert x.flags["C_CONTIGUOUS"]
        return x.ctypes.data
    return x.data_ptr()          # torch tensor


class Sim:
    """One simulator handle.  Method names mirror the C-ABI (ng_ prefix dropped)."""

    def __init__(self, dt_ms: float = 0.1, ring_slots: int = 64, seed: int = 1, record_spikes: bool = True,
                 max_recorded_spikes: int = 1 << 22, debug_input: bool = False, device: int = 0,
                 torch_alloc: bool = True, rank: int = 0, world: int = 1, stream=None):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("paper_2007_14236_b200 needs a CUDA device; there is no CPU fallback")
        self._L = load_library()
        self._torch = torch
        self.device = device
        self.dt_ms, self.D, self.seed = dt_ms, ring_slots, seed
        self.n_ports = 1                          # 2 as soon as an AdEx population is created
        self.stream = stream if stream is not None else torch.cuda.Stream(device=device)
        self.rank, self.world = rank, world
        self._tensors = {}
        self._alloc_struct = None
        if torch_alloc:
            def _alloc(nbytes, _user):
                try:
                    t = torch.empty(int(nbytes), dtype=torch.uint8, device=f"cuda:{device}")
                except Exception:
                    return None
                self._tensors[t.data_ptr()] = t
                return t.data_ptr()

            def _free(ptr, _user):
                self._tensors.pop(ptr, None)

            self._alloc_cb, self._free_cb = _ALLOC_FN(_alloc), _FREE_FN(_free)
            self._alloc_struct = NgAllocator(self._alloc_cb, self._free_cb, None)
        flags = (NG_RECORD_SPIKES if record_spikes else 0) | (NG_DEBUG_INPUT if debug_input else 0)
        cfg = NgConfig(dt_ms, ring_slots, flags, seed, max_recorded_spikes if record_spikes else 0, device, 0)
        h = C.c_void_p()
        rc = self._L.ng_create(C.byref(cfg), C.byref(self._alloc_struct) if self._alloc_struct else None,
                               C.c_void_p(self.stream.cuda_stream), C.byref(h))
        if rc != NG_OK:
            raise NgError(rc, "ng_create failed")
        self._h = h
        if world > 1:
            self._chk(self._L.ng_set_shard(self._h, rank, world))

    # ---- lifetime -------------------------------------------------------------------------------------------
    def close(self):
        if getattr(self, "_h", None):
            self._L.ng_destroy(self._h)
            self._h = None
            self._tensors.clear()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _chk(self, rc, allow=()):
        if rc != NG_OK and rc not in allow:
            raise NgError(rc, self._L.ng_last_error(self._h).decode())
        return rc

    # ---- network description --------------------------------------------------------------------------------
    def create_population(self, n: int, params: dict) -> int:
        """params: LIF dict (ng_lif_params fields) or, with params["model"] == "adex", an AdEx dict (ng_adex_params)."""
        first = C.c_int32()
        if params.get("model") == "adex":
            p = _adex(params)
            self._chk(self._L.ng_create_population_adex(self._h, n, C.byref(p), C.byref(first)))
            self.n_ports = 2
        else:
            p = _lif(params)
            self._chk(self._L.ng_create_population(self._h, n, C.byref(p), C.byref(first)))
        return first.value

    def connect_fixed_indegree(self, src_first, src_n, tgt_first, tgt_n, K, weight, delay, port: int = 0):
        w, d = _dist(weight), _dist(delay)
        self._chk(self._L.ng_connect_fixed_indegree_port(self._h, src_first, src_n, tgt_first, tgt_n, K,
                                                         C.byref(w), C.byref(d), port))

    def connect_fixed_outdegree(self, src_first, src_n, tgt_first, tgt_n, K, weight, delay, port: int = 0):
        w, d = _dist(weight), _dist(delay)
        self._chk(self._L.ng_connect_fixed_outdegree_port(self._h, src_first, src_n, tgt_first, tgt_n, K,
                                                          C.byref(w), C.byref(d), port))

    def set_bypass(self, bypass: bool, inject_fraction: float = 0.0):
        self._chk(self._L.ng_set_bypass(self._h, int(bypass), float(inject_fraction)))

    def set_option(self, option: int, value: int):
        self._chk(self._L.ng_set_option(self._h, option, int(value)))

    def prepare(self):
        self._chk(self._L.ng_prepare(self._h))

    # ---- state ----------------------------------------------------------------------------------------------
    def stats(self) -> NgStats:
        st = NgStats()
        self._chk(self._L.ng_get_stats(self._h, C.byref(st)))
        return st

    @property
    def n_neurons(self) -> int:
        return int(self.stats().n_neurons)

    @property
    def n_connections(self) -> int:
        return int(self.stats().n_connections)

    @property
    def n_sources(self) -> int:
        """Neurons of the whole network (= n_neurons on one GPU): rows of the connection structure."""
        return int(self.stats().n_sources)

    # ---- target-sharded multi-GPU ---------------------------------------------------------------------------
    def exchange_handle(self):
        """(64-byte CUDA IPC handle, device pointer) of this handle's spike-exchange receive buffer."""
        h = (C.c_ubyte * 64)()
        p = C.c_void_p()
        self._chk(self._L.ng_exchange_handle(self._h, h, C.byref(p)))
        return bytes(h), p.value

    def exchange_attach(self, peer_rank: int, ipc_handle: bytes | None = None, ptr: int | None = None):
        buf = (C.c_ubyte * 64).from_buffer_copy(ipc_handle) if ipc_handle is not None else None
        self._chk(self._L.ng_exchange_attach(self._h, peer_rank, buf, C.c_void_p(ptr) if ptr is not None else None))

    def shard_phase(self, phase: int):
        self._chk(self._L.ng_shard_phase(self._h, phase))

    def set_state(self, field: int, data, first: int = 0):
        """data: numpy array or torch tensor (host or device) of the field's element type."""
        if field == FIELD_STEP:
            a = np.asarray([data], dtype=np.int64)
        elif isinstance(data, np.ndarray) or not hasattr(data, "data_ptr"):
            a = np.ascontiguousarray(data, dtype=np.int32 if field == FIELD_REFR else np.float32)
        else:
            a = data.contiguous()
        n = a.size if isinstance(a, np.ndarray) else a.numel()
        self._chk(self._L.ng_set_state(self._h, field, _ptr(a), n, first))

    def get_state(self, field: int, n: int | None = None, first: int = 0, out=None):
        if field == FIELD_STEP:
            a = np.zeros(1, np.int64)
            self._chk(self._L.ng_get_state(self._h, field, a.ctypes.data, 1, 0))
            return int(a[0])
        if out is None:
            if n is None:
                n = self.n_neurons * (self.D * self.n_ports if field == FIELD_RING else
                                      self.n_ports if field == FIELD_LAST_INPUT else 1) - first
            out = np.empty(n, np.int32 if field == FIELD_REFR else np.float32)
        cnt = out.size if isinstance(out, np.ndarray) else out.numel()
        self._chk(self._L.ng_get_state(self._h, field, _ptr(out), cnt, first))
        return out

    # ---- run ------------------------------------------------------------------------------------------------
    def simulate(self, n_steps: int, allow_overflow: bool = False):
        return self._chk(self._L.ng_simulate(self._h, n_steps), allow=(NG_ERR_OVERFLOW,) if allow_overflow else ())

    def get_spikes(self, steps_out=None, ids_out=None):
        """(steps, ids) of every recorded spike as host int32 arrays; drains the device record."""
        cnt = C.c_int64()
        self._chk(self._L.ng_get_spikes(self._h, None, None, 0, C.byref(cnt)))
        n = cnt.value
        steps = steps_out if steps_out is not None else np.empty(n, np.int32)
        ids = ids_out if ids_out is not None else np.empty(n, np.int32)
        cap = min(n, steps.size if isinstance(steps, np.ndarray) else steps.numel())
        if cap > 0:
            self._chk(self._L.ng_get_spikes(self._h, _ptr(steps), _ptr(ids), cap, C.byref(cnt)))
        return steps[:cap], ids[:cap]

    def enable_statistics(self, start_step: int = 0, bin_steps: int = 20, sample_per_pop: int = 200, max_bins: int = 8192):
        self._chk(self._L.ng_enable_statistics(self._h, start_step, bin_steps, sample_per_pop, max_bins))

    def rate_cv(self):
        """(rate_hz[N], cv_isi[N]) computed on the device from the spike-time accumulators."""
        n = self.n_neurons
        rate = np.empty(n, np.float32); cv = np.empty(n, np.float32)
        self._chk(self._L.ng_get_rate_cv(self._h, rate.ctypes.data, cv.ctypes.data, n))
        return rate, cv

    def correlations(self, population: int) -> np.ndarray:
        """Pearson correlation matrix [ns, ns] of the binned spike trains of the population's sample."""
        ns, nb = C.c_int32(), C.c_int32()
        self._chk(self._L.ng_get_correlations(self._h, population, None, 0, C.byref(ns), C.byref(nb)))
        out = np.empty((ns.value, ns.value), np.float32)
        if ns.value and nb.value:
            self._chk(self._L.ng_get_correlations(self._h, population, out.ctypes.data, out.size, C.byref(ns), C.byref(nb)))
        return out

    def trace(self) -> np.ndarray:
        """ng_get_trace: uint64 ns stamps [64 steps][blocks][8] of the last persistent launch (OPT_TRACE)."""
        cnt, blocks = C.c_int64(), C.c_int32()
        self._chk(self._L.ng_get_trace(self._h, None, 0, C.byref(cnt), C.byref(blocks)))
        out = np.zeros(cnt.value, np.uint64)
        self._chk(self._L.ng_get_trace(self._h, out.ctypes.data, cnt.value, C.byref(cnt), C.byref(blocks)))
        return out.reshape(64, blocks.value, -1)

    def last_spikes(self) -> np.ndarray:
        cnt = C.c_int64()
        self._chk(self._L.ng_get_last_spikes(self._h, None, 0, C.byref(cnt)))
        ids = np.empty(cnt.value, np.int32)
        if cnt.value:
            self._chk(self._L.ng_get_last_spikes(self._h, ids.ctypes.data, cnt.value, C.byref(cnt)))
        return ids

    # ---- connection structure read-back (parity checks) --------------------------------------------------------
    def row_offsets(self) -> np.ndarray:
        out = np.empty(self.n_sources + 1, np.int64)
        self._chk(self._L.ng_copy_row_offsets(self._h, out.ctypes.data))
        return out

    def group_offsets(self) -> np.ndarray:
        out = np.empty((self.n_sources, self.D + 1), np.uint32)
        self._chk(self._L.ng_copy_group_offsets(self._h, out.ctypes.data))
        return out

    def records(self, first: int = 0, count: int | None = None):
        if count is None:
            count = int(self.stats().n_records_padded) - first
        tgt = np.empty(count, np.int32); w = np.empty(count, np.float32); d = np.empty(count, np.uint8)
        self._chk(self._L.ng_copy_records(self._h, first, count, tgt.ctypes.data, w.ctypes.data, d.ctypes.data))
        return tgt, w, d

    def connections_of(self, src_id: int):
        cnt = C.c_int64()
        self._chk(self._L.ng_get_connections(self._h, src_id, None, None, None, 0, C.byref(cnt)))
        n = cnt.value
        tgt = np.empty(n, np.int32); w = np.empty(n, np.float32); d = np.empty(n, np.uint8)
        if n:
            self._chk(self._L.ng_get_connections(self._h, src_id, tgt.ctypes.data, w.ctypes.data, d.ctypes.data, n,
                                                 C.byref(cnt)))
        return tgt, w, d


def shard_range(n_neurons: int, rank: int, world: int):
    """ng_shard_range: (first id, count) of the neurons rank `rank` of `world` owns.  Pure host arithmetic."""
    first, n = C.c_int32(), C.c_int32()
    rc = load_library().ng_shard_range(n_neurons, rank, world, C.byref(first), C.byref(n))
    if rc != NG_OK:
        raise NgError(rc, "ng_shard_range: bad arguments")
    return first.value, n.value


def connect_peers(sim: "Sim", dist=None, group=None):
    """Multi-process plumbing of the spike exchange: all-gather the ranks' 64-byte IPC handles with torch.distributed
    (any backend) and map every peer's receive buffer.  Marshalling only — the exchange itself runs in the kernels."""
    import torch.distributed as td
    dist = dist or td
    mine, _ = sim.exchange_handle()
    handles = [None] * sim.world
    dist.all_gather_object(handles, mine, group=group)
    for q, h in enumerate(handles):
        if q != sim.rank:
            sim.exchange_attach(q, ipc_handle=h)


class ShardGroup:
    """All `world` shards of one network as handles of ONE process on ONE device and ONE stream (tests; a box with fewer
    GPUs than ranks).  Steps are issued half by half over all shards (ng_shard_phase), so no kernel ever waits for another.
    Exposes the calls of `Sim` the parity helpers use, with global ids and whole-network arrays."""

    def __init__(self, world: int, dt_ms: float = 0.1, ring_slots: int = 64, seed: int = 1, device: int = 0, **kw):
        import torch
        self.stream = torch.cuda.Stream(device=device)
        self.world, self.D = world, ring_slots
        self.shards = [Sim(dt_ms, ring_slots, seed, device=device, rank=r, world=world, stream=self.stream, **kw) for r in range(world)]

    # network description: the same calls on every shard
    def create_population(self, n, params):
        return [g.create_population(n, params) for g in self.shards][0]

    def connect_fixed_indegree(self, *a, **k):
        for g in self.shards:
            g.connect_fixed_indegree(*a, **k)

    def connect_fixed_outdegree(self, *a, **k):
        for g in self.shards:
            g.connect_fixed_outdegree(*a, **k)

    def set_bypass(self, *a):
        for g in self.shards:
            g.set_bypass(*a)

    def set_option(self, option, value):
        for g in self.shards:
            g.set_option(option, value)

    def prepare(self):
        for g in self.shards:
            g.prepare()
        ptrs = [g.exchange_handle()[1] for g in self.shards]
        for g in self.shards:
            for q, p in enumerate(ptrs):
                if q != g.rank:
                    g.exchange_attach(q, ptr=p)
        self.ranges = [(int(g.stats().id_first), int(g.stats().n_neurons)) for g in self.shards]
        self.n_ports = self.shards[0].n_ports

    @property
    def n_neurons(self):
        return sum(n for _, n in self.ranges)

    def stats(self):
        return [g.stats() for g in self.shards]

    def simulate(self, n_steps: int):
        for _ in range(n_steps):
            for g in self.shards:
                g.shard_phase(0)
            for g in self.shards:
                g.shard_phase(1)
        self._torch_sync()

    def _torch_sync(self):
        self.stream.synchronize()

    def set_state(self, field, data, first: int = 0):
        if field == FIELD_STEP:
            for g in self.shards:
                g.set_state(field, data)
            return
        a = np.ascontiguousarray(data)
        assert first == 0 and field != FIELD_RING
        for g, (f0, n) in zip(self.shards, self.ranges):
            g.set_state(field, a[f0:f0 + n])

    def get_state(self, field, n=None, first: int = 0):
        if field == FIELD_STEP:
            vals = {g.get_state(field) for g in self.shards}
            assert len(vals) == 1
            return vals.pop()
        parts = [g.get_state(field) for g in self.shards]
        if field in (FIELD_RING, FIELD_LAST_INPUT):          # [slots][ports][local N] per shard -> [slots][ports][N]
            rows = [p.reshape(-1, nloc) for p, (_, nloc) in zip(parts, self.ranges)]
            return np.concatenate(rows, axis=1).reshape(-1)
        return np.concatenate(parts)

    def last_spikes(self):
        ids = [np.sort(g.last_spikes()) for g in self.shards]
        for other in ids[1:]:
            assert np.array_equal(ids[0], other), "shards disagree on the spike array"
        return ids[0]

    def get_spikes(self):
        rec = [g.get_spikes() for g in self.shards]
        key0 = np.lexsort((rec[0][1], rec[0][0]))
        for s_, i_ in rec[1:]:
            k = np.lexsort((i_, s_))
            assert np.array_equal(rec[0][0][key0], s_[k]) and np.array_equal(rec[0][1][key0], i_[k]), "shards disagree on the spike record"
        return rec[0][0][key0], rec[0][1][key0]

    def connections(self):
        """(src, tgt, weight, delay) of the whole network with GLOBAL target ids, concatenated over the shards (padding removed)."""
        out = []
        for g, (f0, nloc) in zip(self.shards, self.ranges):
            ro = g.row_offsets(); tgt, w, d = g.records()
            src = np.repeat(np.arange(ro.size - 1, dtype=np.int32), np.diff(ro))
            keep = tgt >= 0
            port = tgt[keep] // nloc
            out.append((src[keep], (tgt[keep] % nloc) + f0, w[keep], d[keep], port))
        return tuple(np.concatenate([o[k] for o in out]) for k in range(5))

    def close(self):
        for g in self.shards:
            g.close()
