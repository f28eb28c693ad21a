"""oracle — TEST INFRASTRUCTURE, not the product.

ctypes harness around ``oracle/oracle.cpp`` (plain fp64 CPU restatement of the hot path of
arXiv 2007.14236, see that file's header for the passages it follows and its pins).

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` leg may import this package.  It imports nothing from
``paper_2007_14236_b200`` and the product imports nothing from here.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "oracle.cpp")
_HDR = os.path.join(_HERE, "oracle_adex.hpp")
_LIB = os.path.join(_HERE, "liboracle.so")

FIELD_V, FIELD_I_SYN, FIELD_REFR, FIELD_RING, FIELD_STEP = 0, 1, 2, 3, 4
FIELD_W, FIELD_G_EX, FIELD_Y_EX, FIELD_G_IN, FIELD_Y_IN, FIELD_H_INT = 6, 7, 8, 9, 10, 11        # AdEx state
DIST_CONST, DIST_NORMAL_CLIPPED, DIST_UNIFORM_INT = 0, 1, 2
RULE_FIXED_INDEGREE, RULE_FIXED_OUTDEGREE = 0, 1


def build(force: bool = False) -> str:
    """Compile oracle.cpp with g++ (no fast-math, no FMA contraction)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < max(os.path.getmtime(_SRC), os.path.getmtime(_HDR)):
        cmd = ["g++", "-O2", "-std=c++17", "-ffp-contract=off", "-fno-fast-math", "-shared", "-fPIC",
               _SRC, "-o", _LIB]
        subprocess.check_call(cmd)
    return _LIB


class _LifParams(C.Structure):
    _fields_ = [(k, C.c_double) for k in
                ("C_m", "tau_m", "tau_syn", "E_L", "V_th", "V_reset", "t_ref_ms", "I_e",
                 "poisson_rate_hz", "poisson_weight")]


_ADEX_SCALARS = ("C_m", "g_L", "E_L", "V_T", "Delta_T", "tau_w", "a", "b", "V_reset", "V_peak", "E_ex", "E_in", "tau_syn",
                 "I_e", "poisson_rate_hz", "poisson_weight")


class _AdexParams(C.Structure):
    _fields_ = [(k, C.c_double) for k in _ADEX_SCALARS] + [("tol", C.c_double * 6), ("h_min", C.c_double)]


def _adex(params: dict) -> _AdexParams:
    p = _AdexParams(**{k: float(params.get(k, 0.0)) for k in _ADEX_SCALARS})
    for i, t in enumerate(params["tol"]):
        p.tol[i] = float(t)
    p.h_min = float(params["h_min"])
    return p


class _Dist(C.Structure):
    _fields_ = [("kind", C.c_int32), ("pad", C.c_int32), ("a", C.c_double), ("b", C.c_double),
                ("lo", C.c_double), ("hi", C.c_double)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        L.orc_create.restype = C.c_void_p
        L.orc_create.argtypes = [C.c_double, C.c_int32, C.c_uint64]
        L.orc_destroy.argtypes = [C.c_void_p]
        L.orc_last_error.restype = C.c_char_p
        L.orc_last_error.argtypes = [C.c_void_p]
        L.orc_set_bypass.argtypes = [C.c_void_p, C.c_int32, C.c_double]
        L.orc_create_population.argtypes = [C.c_void_p, C.c_int32, C.POINTER(_LifParams), C.POINTER(C.c_int32)]
        L.orc_connect.argtypes = [C.c_void_p] + [C.c_int32] * 6 + [C.POINTER(_Dist), C.POINTER(_Dist)]
        L.orc_connect_port.argtypes = [C.c_void_p] + [C.c_int32] * 6 + [C.POINTER(_Dist), C.POINTER(_Dist), C.c_int32]
        L.orc_create_population_adex.argtypes = [C.c_void_p, C.c_int32, C.POINTER(_AdexParams), C.POINTER(C.c_int32)]
        L.orc_adex_rhs.argtypes = [C.POINTER(_AdexParams), C.c_void_p, C.c_void_p]
        L.orc_adex_step.argtypes = [C.POINTER(_AdexParams), C.c_void_p, C.c_void_p, C.c_double]
        L.orc_num_ports.argtypes = [C.c_void_p]
        L.orc_prepare.argtypes = [C.c_void_p]
        L.orc_num_connections.restype = C.c_int64
        L.orc_num_connections.argtypes = [C.c_void_p]
        L.orc_num_neurons.argtypes = [C.c_void_p]
        L.orc_get_connections.argtypes = [C.c_void_p] + [C.c_void_p] * 5
        L.orc_draw_connection.argtypes = [C.c_void_p, C.c_int32, C.c_int32, C.c_int32, C.c_void_p, C.c_void_p]
        L.orc_poisson_count.argtypes = [C.c_void_p, C.c_int32, C.c_int64]
        L.orc_set_state.argtypes = [C.c_void_p, C.c_int32, C.c_void_p, C.c_int64, C.c_int64]
        L.orc_get_state.argtypes = [C.c_void_p, C.c_int32, C.c_void_p, C.c_int64, C.c_int64]
        L.orc_simulate.argtypes = [C.c_void_p, C.c_int64, C.c_int32]
        L.orc_num_spikes.restype = C.c_int64
        L.orc_num_spikes.argtypes = [C.c_void_p]
        L.orc_get_spikes.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int64, C.c_int32]
        L.orc_num_last_spikes.restype = C.c_int64
        L.orc_num_last_spikes.argtypes = [C.c_void_p]
        L.orc_get_last_spikes.argtypes = [C.c_void_p, C.c_void_p]
        L.orc_num_events.restype = C.c_uint64
        L.orc_num_events.argtypes = [C.c_void_p]
        L.orc_philox4x32_10.argtypes = [C.c_uint32, C.c_uint32, C.c_void_p, C.c_void_p]
        L.orc_propagators.argtypes = [C.POINTER(_LifParams), C.c_double, C.c_void_p]
        L.orc_poisson_table.argtypes = [C.c_double, C.c_void_p, C.c_int32]
        _lib = L
    return _lib


def _lif(params: dict) -> _LifParams:
    return _LifParams(**{k: float(params.get(k, 0.0)) for k, _ in _LifParams._fields_})


def _dist(d) -> _Dist:
    """d = ("const", a) | ("normal", mean, sd[, lo, hi]) | ("uniform_int", lo, hi)."""
    kind = d[0]
    if kind == "const":
        return _Dist(DIST_CONST, 0, float(d[1]), 0.0, 0.0, 0.0)
    if kind == "normal":
        lo = float(d[3]) if len(d) > 3 else -np.inf
        hi = float(d[4]) if len(d) > 4 else np.inf
        return _Dist(DIST_NORMAL_CLIPPED, 0, float(d[1]), float(d[2]), lo, hi)
    if kind == "uniform_int":
        return _Dist(DIST_UNIFORM_INT, 0, 0.0, 0.0, float(d[1]), float(d[2]))
    raise ValueError(kind)


def philox4x32_10(key_lo: int, key_hi: int, ctr) -> np.ndarray:
    c = np.asarray(ctr, dtype=np.uint32)
    out = np.zeros(4, dtype=np.uint32)
    lib().orc_philox4x32_10(key_lo, key_hi, c.ctypes.data, out.ctypes.data)
    return out


def propagators(params: dict, h: float) -> np.ndarray:
    """(P11, P22, P21, P20) for step h [ms]."""
    out = np.zeros(4)
    p = _lif(params)
    lib().orc_propagators(C.byref(p), h, out.ctypes.data)
    return out


def adex_rhs(params: dict, y) -> np.ndarray:
    """Right-hand side of the AdEx system (oracle_adex.hpp): y = (V, w, g_ex, y_ex, g_in, y_in)."""
    a = np.ascontiguousarray(y, dtype=np.float64); f = np.zeros(6)
    p = _adex(params)
    lib().orc_adex_rhs(C.byref(p), a.ctypes.data, f.ctypes.data)
    return f


def adex_step(params: dict, y, h_int: float, h_step: float):
    """One time step of the adaptive Cash-Karp integrator: returns (y', h_int', spiked)."""
    a = np.array(y, dtype=np.float64); h = np.array([h_int], dtype=np.float64)
    p = _adex(params)
    spk = lib().orc_adex_step(C.byref(p), a.ctypes.data, h.ctypes.data, float(h_step))
    return a, float(h[0]), bool(spk)


def poisson_table(lam: float) -> np.ndarray:
    out = np.zeros(64, dtype=np.uint32)
    n = lib().orc_poisson_table(lam, out.ctypes.data, 64)
    if n < 0:
        raise ValueError("lambda too large")
    return out[:n].copy()


class Oracle:
    """Same method names as the product binding (duck-typed by the workload recipes)."""

    def __init__(self, dt_ms: float = 0.1, ring_slots: int = 64, seed: int = 1):
        self._L = lib()
        self._h = self._L.orc_create(dt_ms, ring_slots, seed)
        self.dt_ms, self.D, self.seed = dt_ms, ring_slots, seed

    def __del__(self):
        if getattr(self, "_h", None):
            self._L.orc_destroy(self._h)
            self._h = None

    def _chk(self, rc):
        if rc != 0:
            raise RuntimeError(f"oracle error {rc}: {self._L.orc_last_error(self._h).decode()}")

    def set_bypass(self, bypass: bool, inject_fraction: float = 0.0):
        self._chk(self._L.orc_set_bypass(self._h, int(bypass), inject_fraction))

    def create_population_adex(self, n: int, params: dict) -> int:
        first = C.c_int32()
        p = _adex(params)
        self._chk(self._L.orc_create_population_adex(self._h, n, C.byref(p), C.byref(first)))
        return first.value

    @property
    def n_ports(self) -> int:
        return self._L.orc_num_ports(self._h)

    def create_population(self, n: int, params: dict) -> int:
        if params.get("model") == "adex":
            return self.create_population_adex(n, params)
        first = C.c_int32()
        p = _lif(params)
        self._chk(self._L.orc_create_population(self._h, n, C.byref(p), C.byref(first)))
        return first.value

    def connect_fixed_indegree(self, src_first, src_n, tgt_first, tgt_n, K, weight, delay, port: int = 0):
        w, d = _dist(weight), _dist(delay)
        self._chk(self._L.orc_connect_port(self._h, RULE_FIXED_INDEGREE, src_first, src_n, tgt_first, tgt_n, K,
                                           C.byref(w), C.byref(d), port))

    def connect_fixed_outdegree(self, src_first, src_n, tgt_first, tgt_n, K, weight, delay, port: int = 0):
        w, d = _dist(weight), _dist(delay)
        self._chk(self._L.orc_connect_port(self._h, RULE_FIXED_OUTDEGREE, src_first, src_n, tgt_first, tgt_n, K,
                                           C.byref(w), C.byref(d), port))

    def prepare(self):
        self._chk(self._L.orc_prepare(self._h))

    @property
    def n_neurons(self) -> int:
        return self._L.orc_num_neurons(self._h)

    @property
    def n_connections(self) -> int:
        return self._L.orc_num_connections(self._h)

    def get_connections(self):
        """Canonical (src, tgt, w, delay, row_off), ordered by (src, delay, tgt, call, k)."""
        S, N = self.n_connections, self.n_neurons
        src = np.empty(S, np.int32); tgt = np.empty(S, np.int32)
        w = np.empty(S, np.float32); d = np.empty(S, np.uint8); ro = np.empty(N + 1, np.int64)
        self._chk(self._L.orc_get_connections(self._h, src.ctypes.data, tgt.ctypes.data, w.ctypes.data,
                                              d.ctypes.data, ro.ctypes.data))
        return src, tgt, w, d, ro

    def draw_connection(self, call: int, endpoint: int, k: int):
        out = np.zeros(3, np.int32); w = np.zeros(1, np.float32)
        self._chk(self._L.orc_draw_connection(self._h, call, endpoint, k, out.ctypes.data, w.ctypes.data))
        return int(out[0]), int(out[1]), int(out[2]), np.float32(w[0])

    def poisson_count(self, i: int, n: int) -> int:
        return self._L.orc_poisson_count(self._h, i, n)

    def set_state(self, field: int, data, first: int = 0):
        if field == FIELD_STEP:
            a = np.asarray([data], dtype=np.int64)
        elif field == FIELD_REFR:
            a = np.ascontiguousarray(data, dtype=np.int32)
        else:
            a = np.ascontiguousarray(data, dtype=np.float64)
        self._chk(self._L.orc_set_state(self._h, field, a.ctypes.data, a.size, first))

    def get_state(self, field: int, n: int | None = None, first: int = 0):
        if field == FIELD_STEP:
            a = np.zeros(1, np.int64)
            self._chk(self._L.orc_get_state(self._h, field, a.ctypes.data, 1, 0))
            return int(a[0])
        if n is None:
            n = self.n_neurons * (self.D * self.n_ports if field == FIELD_RING else 1) - first
        a = np.empty(n, np.int32 if field == FIELD_REFR else np.float64)
        self._chk(self._L.orc_get_state(self._h, field, a.ctypes.data, n, first))
        return a

    def simulate(self, n_steps: int, record: bool = True):
        self._chk(self._L.orc_simulate(self._h, n_steps, int(record)))

    def get_spikes(self, drain: bool = True):
        n = self._L.orc_num_spikes(self._h)
        steps = np.empty(n, np.int32); ids = np.empty(n, np.int32)
        self._L.orc_get_spikes(self._h, steps.ctypes.data, ids.ctypes.data, n, int(drain))
        return steps, ids

    def last_spikes(self) -> np.ndarray:
        n = self._L.orc_num_last_spikes(self._h)
        ids = np.empty(n, np.int32)
        self._L.orc_get_last_spikes(self._h, ids.ctypes.data)
        return ids

    @property
    def n_events(self) -> int:
        return self._L.orc_num_events(self._h)
