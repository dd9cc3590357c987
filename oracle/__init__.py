"""CPU ORACLE for the network-construction hot path of arXiv 2306.09855 -- TEST INFRASTRUCTURE.

Only ``tests/``, ``__graft_entry__.smoke()`` and the ``cpu_baseline`` / ``--impl reference`` legs
of ``bench.py`` may import this package.  It never imports the product package
(``paper_2306_09855_b200``) and the product never imports it.

``oracle.cpp`` is the oracle itself (plain single-threaded fp64 C++, written from PAPER.md);
this module only compiles it with g++ and marshals arguments through ctypes.
"""
from __future__ import annotations

import ctypes as C
import math
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_LIB_PATH = _HERE / "liboracle.so"

ONE_TO_ONE, ALL_TO_ALL, FIXED_INDEGREE, FIXED_OUTDEGREE, FIXED_TOTAL_NUMBER, PAIRWISE_BERNOULLI = range(6)
RULES = {
    "one_to_one": ONE_TO_ONE,
    "all_to_all": ALL_TO_ALL,
    "fixed_indegree": FIXED_INDEGREE,
    "fixed_outdegree": FIXED_OUTDEGREE,
    "fixed_total_number": FIXED_TOTAL_NUMBER,
    "pairwise_bernoulli": PAIRWISE_BERNOULLI,
}
OK, ERR_INVALID_ARG, ERR_STATE, ERR_CAPACITY, ERR_OOM = 0, -1, -2, -3, -4


def build(force: bool = False) -> Path:
    """Compile oracle.cpp + delivery.cpp + copass.cpp -> liboracle.so (g++ -O2 -ffp-contract=off)."""
    srcs = [_HERE / "oracle.cpp", _HERE / "oracle.h", _HERE / "delivery.cpp", _HERE / "delivery.h",
            _HERE / "copass.cpp", _HERE / "copass.h"]
    if not force and _LIB_PATH.exists() and all(_LIB_PATH.stat().st_mtime >= s.stat().st_mtime for s in srcs):
        return _LIB_PATH
    tmp = _LIB_PATH.with_suffix(f".so.tmp{os.getpid()}")
    cmd = ["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-fPIC", "-shared", "-Wall", "-Wextra",
           "-o", str(tmp), str(_HERE / "oracle.cpp"), str(_HERE / "delivery.cpp"), str(_HERE / "copass.cpp")]
    subprocess.run(cmd, check=True)
    os.replace(tmp, _LIB_PATH)
    return _LIB_PATH


class _Config(C.Structure):
    _fields_ = [("block_size", C.c_uint64), ("dt_ms", C.c_double)]


class _RuleParams(C.Structure):
    _fields_ = [("degree_or_total", C.c_uint64), ("p", C.c_double)]


class _Dist(C.Structure):
    _fields_ = [("mean", C.c_double), ("sd", C.c_double), ("lo", C.c_double), ("hi", C.c_double)]


class _SynSpec(C.Structure):
    _fields_ = [("weight", _Dist), ("delay_ms", _Dist)]


class _Range(C.Structure):
    _fields_ = [("first", C.c_uint32), ("count", C.c_uint32)]


class _ConnView(C.Structure):
    _fields_ = [("source", C.POINTER(C.c_uint32)), ("target", C.POINTER(C.c_uint32)),
                ("weight", C.POINTER(C.c_float)), ("delay", C.POINTER(C.c_uint16)),
                ("perm", C.POINTER(C.c_uint32)), ("boundary", C.POINTER(C.c_uint8)), ("n", C.c_uint64)]


class _IndexView(C.Structure):
    _fields_ = [("src_offsets", C.POINTER(C.c_uint32)), ("group_count", C.POINTER(C.c_uint32)),
                ("group_ptr", C.POINTER(C.c_uint32)), ("group_start", C.POINTER(C.c_uint32)),
                ("group_delay", C.POINTER(C.c_uint16)), ("n_nodes", C.c_uint32), ("total_groups", C.c_uint32)]


class _Synapse(C.Structure):
    _fields_ = [("source", C.c_uint32), ("target", C.c_uint32), ("weight", C.c_float),
                ("delay", C.c_uint16), ("boundary", C.c_uint8), ("accepted", C.c_uint8),
                ("z0", C.c_double), ("z1", C.c_double), ("x", C.c_double)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(str(build()))
        P = C.POINTER
        L.oc_create.argtypes = [P(_Config), P(C.c_void_p)]
        L.oc_destroy.argtypes = [C.c_void_p]
        L.oc_create_population.argtypes = [C.c_void_p, C.c_uint32, P(C.c_uint32)]
        L.oc_connect.argtypes = [C.c_void_p, _Range, _Range, C.c_int, P(_RuleParams), P(_SynSpec), C.c_uint64]
        L.oc_finalize.argtypes = [C.c_void_p]
        L.oc_num_connections.argtypes = [C.c_void_p, P(C.c_uint64)]
        L.oc_num_nodes.argtypes = [C.c_void_p, P(C.c_uint32)]
        L.oc_num_blocks.argtypes = [C.c_void_p, P(C.c_uint64)]
        L.oc_block_slot.argtypes = [C.c_void_p, C.c_uint64, P(C.c_uint64), P(C.c_uint64)]
        L.oc_get_connections.argtypes = [C.c_void_p, C.c_int, P(_ConnView)]
        L.oc_get_index.argtypes = [C.c_void_p, P(_IndexView)]
        L.oc_degree_histogram.argtypes = [C.c_void_p, C.c_int, P(P(C.c_uint32)), P(C.c_uint32)]
        L.oc_philox4x32_10.argtypes = [P(C.c_uint32), P(C.c_uint32), P(C.c_uint32)]
        L.oc_philox4x32_10.restype = None
        L.oc_bounded.argtypes = [C.c_uint32, C.c_uint32]
        L.oc_bounded.restype = C.c_uint32
        L.oc_bernoulli_threshold.argtypes = [C.c_double]
        L.oc_bernoulli_threshold.restype = C.c_uint64
        L.oc_bernoulli_trial_word.argtypes = [C.c_uint64, C.c_uint32, C.c_uint64]
        L.oc_bernoulli_trial_word.restype = C.c_uint32
        L.oc_eval_synapse.argtypes = [_Range, _Range, C.c_int, P(_RuleParams), P(_SynSpec), C.c_uint64,
                                      C.c_uint32, C.c_double, C.c_uint64, P(_Synapse)]
        _lib = L
    return _lib


def _dist(d) -> _Dist:
    mean, sd, lo, hi = d
    return _Dist(float(mean), float(sd), float(lo), float(hi))


def _syn(weight, delay_ms) -> _SynSpec:
    return _SynSpec(_dist(weight), _dist(delay_ms))


def _np(ptr, n, dtype):
    if n == 0:
        return np.zeros(0, dtype=dtype)
    return np.ctypeslib.as_array(ptr, shape=(int(n),)).view(dtype)


class OracleError(RuntimeError):
    def __init__(self, code):
        super().__init__(f"oracle error {code}")
        self.code = code


def philox4x32_10(ctr, key):
    c = (C.c_uint32 * 4)(*ctr)
    k = (C.c_uint32 * 2)(*key)
    o = (C.c_uint32 * 4)()
    lib().oc_philox4x32_10(c, k, o)
    return tuple(int(v) for v in o)


def bounded(word: int, n: int) -> int:
    return int(lib().oc_bounded(word, n))


def bernoulli_threshold(p: float) -> int:
    return int(lib().oc_bernoulli_threshold(p))


def bernoulli_trial_word(seed: int, projection_id: int, q: int) -> int:
    return int(lib().oc_bernoulli_trial_word(seed, projection_id, q))


def eval_synapse(src, tgt, rule, degree_or_total, p, weight, delay_ms, seed, projection_id, dt_ms, idx):
    """One synapse as a pure function of (seed, projection_id, idx); returns a dict."""
    rp = _RuleParams(int(degree_or_total), float(p))
    sp = _syn(weight, delay_ms)
    out = _Synapse()
    rc = lib().oc_eval_synapse(_Range(*src), _Range(*tgt), int(rule), C.byref(rp), C.byref(sp), int(seed),
                               int(projection_id), float(dt_ms), int(idx), C.byref(out))
    if rc != 0:
        raise OracleError(rc)
    return {f: getattr(out, f) for f, _ in _Synapse._fields_}


def eval_synapses(src, tgt, rule, degree_or_total, p, weight, delay_ms, seed, projection_id, dt_ms, idx) -> dict:
    """eval_synapse over an array of indexes (oc_eval_synapse_batch); returns a dict of arrays."""
    idx = np.ascontiguousarray(idx, dtype=np.uint64)
    n = idx.size
    rp = _RuleParams(int(degree_or_total), float(p))
    sp = _syn(weight, delay_ms)
    out = {"source": np.empty(n, np.uint32), "target": np.empty(n, np.uint32), "weight": np.empty(n, np.float32),
           "delay": np.empty(n, np.uint16), "boundary": np.empty(n, np.uint8), "accepted": np.empty(n, np.uint8)}
    L = lib()
    L.oc_eval_synapse_batch.argtypes = [_Range, _Range, C.c_int, C.POINTER(_RuleParams), C.POINTER(_SynSpec), C.c_uint64,
                                        C.c_uint32, C.c_double, C.c_void_p, C.c_uint64] + [C.c_void_p] * 6
    vp = lambda a: a.ctypes.data_as(C.c_void_p)  # noqa: E731
    rc = L.oc_eval_synapse_batch(_Range(*src), _Range(*tgt), int(rule), C.byref(rp), C.byref(sp), int(seed),
                                 int(projection_id), float(dt_ms), vp(idx), n, vp(out["source"]), vp(out["target"]),
                                 vp(out["weight"]), vp(out["delay"]), vp(out["boundary"]), vp(out["accepted"]))
    if rc != 0:
        raise OracleError(rc)
    return out


class Oracle:
    """Same call sequence as the nc_ ABI (create_population / connect / finalize / getters)."""

    def __init__(self, dt_ms: float = 0.1, block_size: int = 0):
        self._h = C.c_void_p()
        cfg = _Config(int(block_size), float(dt_ms))
        rc = lib().oc_create(C.byref(cfg), C.byref(self._h))
        if rc != 0:
            raise OracleError(rc)

    def close(self):
        if self._h:
            lib().oc_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def create_population(self, n: int) -> int:
        first = C.c_uint32()
        rc = lib().oc_create_population(self._h, int(n), C.byref(first))
        if rc != 0:
            raise OracleError(rc)
        return first.value

    def connect_rc(self, src, tgt, rule, degree_or_total=0, p=0.0, weight=(1.0, 0.0, -math.inf, math.inf),
                   delay_ms=(1.0, 0.0, -math.inf, math.inf), seed=0, weights=None, delays=None) -> int:
        """weights / delays: per-connection value arrays (oc_connect_values); None = follow the
        distributions."""
        rp = _RuleParams(int(degree_or_total), float(p))
        sp = _syn(weight, delay_ms)
        if weights is not None or delays is not None:
            sa = None if isinstance(src, tuple) else np.ascontiguousarray(src, dtype=np.uint32)
            ta = None if isinstance(tgt, tuple) else np.ascontiguousarray(tgt, dtype=np.uint32)
            wa = None if weights is None else np.ascontiguousarray(weights, dtype=np.float32)
            da = None if delays is None else np.ascontiguousarray(delays, dtype=np.float64)
            L = lib()
            L.oc_connect_values.argtypes = [C.c_void_p, C.c_void_p, C.c_uint32, _Range, C.c_void_p, C.c_uint32, _Range,
                                            C.c_int, C.c_void_p, C.c_void_p, C.c_uint64, C.c_void_p, C.c_void_p,
                                            C.c_uint64]
            L.oc_connect_values.restype = C.c_int
            vp = lambda a: None if a is None else a.ctypes.data_as(C.c_void_p)
            return int(L.oc_connect_values(self._h, vp(sa), 0 if sa is None else sa.size,
                                           _Range(0, 0) if sa is not None else _Range(*src), vp(ta),
                                           0 if ta is None else ta.size, _Range(0, 0) if ta is not None else _Range(*tgt),
                                           int(rule), C.byref(rp), C.byref(sp), int(seed), vp(wa), vp(da),
                                           (wa if wa is not None else da).size))
        if isinstance(src, tuple) and isinstance(tgt, tuple):
            return int(lib().oc_connect(self._h, _Range(*src), _Range(*tgt), int(rule), C.byref(rp), C.byref(sp),
                                        int(seed)))
        # a side that is not a (first, count) tuple is an explicit array of node ids
        sa = None if isinstance(src, tuple) else np.ascontiguousarray(src, dtype=np.uint32)
        ta = None if isinstance(tgt, tuple) else np.ascontiguousarray(tgt, dtype=np.uint32)
        L = lib()
        L.oc_connect_nodes.argtypes = [C.c_void_p, C.c_void_p, C.c_uint32, _Range, C.c_void_p, C.c_uint32, _Range, C.c_int,
                                       C.c_void_p, C.c_void_p, C.c_uint64]
        L.oc_connect_nodes.restype = C.c_int
        return int(L.oc_connect_nodes(self._h, None if sa is None else sa.ctypes.data_as(C.c_void_p),
                                      0 if sa is None else sa.size, _Range(0, 0) if sa is not None else _Range(*src),
                                      None if ta is None else ta.ctypes.data_as(C.c_void_p),
                                      0 if ta is None else ta.size, _Range(0, 0) if ta is not None else _Range(*tgt),
                                      int(rule), C.byref(rp), C.byref(sp), int(seed)))

    def connect(self, *a, **k):
        rc = self.connect_rc(*a, **k)
        if rc != 0:
            raise OracleError(rc)

    def set_shard(self, first: int, count: int):
        L = lib()
        L.oc_set_shard.argtypes = [C.c_void_p, C.c_uint32, C.c_uint32]
        rc = L.oc_set_shard(self._h, int(first), int(count))
        if rc != 0:
            raise OracleError(rc)

    def set_rule_flags(self, flags: int):
        L = lib()
        L.oc_set_rule_flags.argtypes = [C.c_void_p, C.c_uint32]
        rc = L.oc_set_rule_flags(self._h, int(flags))
        if rc != 0:
            raise OracleError(rc)

    def set_connection_attributes(self, port: int, syn_group: int = 0):
        L = lib()
        L.oc_set_connection_attributes.argtypes = [C.c_void_p, C.c_uint8, C.c_uint8]
        rc = L.oc_set_connection_attributes(self._h, int(port), int(syn_group))
        if rc != 0:
            raise OracleError(rc)

    def read_connection_attributes(self, sorted: bool = False, first: int = 0, count=None):
        L = lib()
        L.oc_read_connection_attributes.argtypes = [C.c_void_p, C.c_int, C.c_uint64, C.c_uint64, C.c_void_p, C.c_void_p]
        if count is None:
            count = self.num_connections() - first
        port, group = np.zeros(count, np.uint8), np.zeros(count, np.uint8)
        rc = L.oc_read_connection_attributes(self._h, 1 if sorted else 0, int(first), int(count),
                                             port.ctypes.data_as(C.c_void_p), group.ctypes.data_as(C.c_void_p))
        if rc != 0:
            raise OracleError(rc)
        return port, group

    def finalize(self):
        rc = lib().oc_finalize(self._h)
        if rc != 0:
            raise OracleError(rc)

    def num_connections(self) -> int:
        n = C.c_uint64()
        lib().oc_num_connections(self._h, C.byref(n))
        return n.value

    def num_nodes(self) -> int:
        n = C.c_uint32()
        lib().oc_num_nodes(self._h, C.byref(n))
        return n.value

    def num_blocks(self) -> int:
        n = C.c_uint64()
        lib().oc_num_blocks(self._h, C.byref(n))
        return n.value

    def block_slot(self, pos: int):
        b, s = C.c_uint64(), C.c_uint64()
        lib().oc_block_slot(self._h, int(pos), C.byref(b), C.byref(s))
        return b.value, s.value

    def projection_starts(self) -> np.ndarray:
        """Creation position at which each projection starts, closed by the current number of connections."""
        L = lib()
        L.oc_get_projection_starts.argtypes = [C.c_void_p, C.POINTER(C.POINTER(C.c_uint64)), C.POINTER(C.c_uint32)]
        p, n = C.POINTER(C.c_uint64)(), C.c_uint32()
        rc = L.oc_get_projection_starts(self._h, C.byref(p), C.byref(n))
        if rc != 0:
            raise OracleError(rc)
        return np.concatenate([_np(p, n.value, np.uint64).astype(np.int64), [self.num_connections()]]).astype(np.int64)

    def connections(self, sorted: bool = False, copy: bool = True) -> dict:
        """Arrays are COPIES (safe to keep after further calls) unless copy=False (views into the oracle's own
        vectors, valid until the next connect / finalize / close -- for networks too large to duplicate)."""
        v = _ConnView()
        rc = lib().oc_get_connections(self._h, 1 if sorted else 0, C.byref(v))
        if rc != 0:
            raise OracleError(rc)
        n = v.n
        cp = (lambda a: a.copy()) if copy else (lambda a: a)
        out = {
            "source": cp(_np(v.source, n, np.uint32)),
            "target": cp(_np(v.target, n, np.uint32)),
            "weight": cp(_np(v.weight, n, np.float32)),
            "delay": cp(_np(v.delay, n, np.uint16)),
            "boundary": cp(_np(v.boundary, n, np.uint8)),
            "n": int(n),
        }
        if sorted:
            out["perm"] = cp(_np(v.perm, n, np.uint32))
        return out

    def index(self) -> dict:
        v = _IndexView()
        rc = lib().oc_get_index(self._h, C.byref(v))
        if rc != 0:
            raise OracleError(rc)
        N, G = v.n_nodes, v.total_groups
        return {
            "src_offsets": _np(v.src_offsets, N + 1, np.uint32).copy(),
            "group_count": _np(v.group_count, N, np.uint32).copy(),
            "group_ptr": _np(v.group_ptr, N + 1, np.uint32).copy(),
            "group_start": _np(v.group_start, G, np.uint32).copy(),
            "group_delay": _np(v.group_delay, G, np.uint16).copy(),
            "n_nodes": int(N),
            "total_groups": int(G),
        }

    def degree_histogram(self, kind: int):
        p = C.POINTER(C.c_uint32)()
        mx = C.c_uint32()
        rc = lib().oc_degree_histogram(self._h, int(kind), C.byref(p), C.byref(mx))
        if rc != 0:
            raise OracleError(rc)
        return _np(p, self.num_nodes(), np.uint32).copy(), mx.value


class Delivery:
    """Spike delivery over a finalized Oracle (delivery.h).  `input` is an fp64 array of n_nodes that
    every step accumulates into."""

    def __init__(self, oracle: "Oracle"):
        L = lib()
        L.oc_delivery_create.argtypes = [C.c_void_p, C.POINTER(C.c_void_p)]
        L.oc_delivery_destroy.argtypes = [C.c_void_p]
        L.oc_delivery_step.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_uint32, C.c_void_p]
        L.oc_delivery_spike_array.argtypes = [C.c_void_p, C.POINTER(C.POINTER(C.c_uint32)),
                                              C.POINTER(C.POINTER(C.c_uint32)), C.POINTER(C.c_uint32)]
        L.oc_delivery_counts.argtypes = [C.c_void_p, C.POINTER(C.c_uint64), C.POINTER(C.c_uint64)]
        self._L, self._oracle = L, oracle  # the oracle context must outlive this object
        self._h = C.c_void_p()
        rc = L.oc_delivery_create(oracle._h, C.byref(self._h))
        if rc != 0:
            raise OracleError(rc)
        self.n_nodes = oracle.num_nodes()
        L.oc_delivery_num_ports.argtypes = [C.c_void_p, C.POINTER(C.c_uint32)]
        np_ = C.c_uint32()
        L.oc_delivery_num_ports(self._h, C.byref(np_))
        self.n_ports = np_.value

    def step(self, nodes, mult, input_f64):
        nodes = np.ascontiguousarray(nodes, dtype=np.uint32)
        m = None if mult is None else np.ascontiguousarray(mult, dtype=np.uint32)
        assert input_f64.dtype == np.float64 and input_f64.size == self.n_nodes * self.n_ports and input_f64.flags.c_contiguous
        rc = self._L.oc_delivery_step(self._h, nodes.ctypes.data_as(C.c_void_p),
                                      None if m is None else m.ctypes.data_as(C.c_void_p), nodes.size,
                                      input_f64.ctypes.data_as(C.c_void_p))
        if rc != 0:
            raise OracleError(rc)

    def spike_array(self):
        g, m, n = C.POINTER(C.c_uint32)(), C.POINTER(C.c_uint32)(), C.c_uint32()
        self._L.oc_delivery_spike_array(self._h, C.byref(g), C.byref(m), C.byref(n))
        return _np(g, n.value, np.uint32).copy(), _np(m, n.value, np.uint32).copy()

    def counts(self):
        b, e = C.c_uint64(), C.c_uint64()
        self._L.oc_delivery_counts(self._h, C.byref(b), C.byref(e))
        return b.value, e.value

    def close(self):
        if self._h:
            self._L.oc_delivery_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


# ---------------------------------------------------------------------------------------------------------------
# COPASS block-sort (copass.h)
# ---------------------------------------------------------------------------------------------------------------
class _CopassInfo(C.Structure):
    _fields_ = [("t", C.c_int64), ("iterations", C.c_uint32), ("last_step", C.c_int32)]


class _CopassStats(C.Structure):
    _fields_ = [("aux_peak", C.c_uint64), ("moved", C.c_uint64), ("partitions", C.c_uint32),
                ("iterations", C.c_uint32), ("last_step_1", C.c_uint32), ("last_step_2", C.c_uint32)]


def copass_partition(keys, start, length, m):
    """oc_copass_partition: keys int64 flat array, subarray i = keys[start[i] : start[i] + length[i]] ascending.
    Returns (m_i uint64[k], t, iterations, last_step)."""
    L = lib()
    L.oc_copass_partition.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_uint32, C.c_uint64, C.c_void_p,
                                      C.POINTER(_CopassInfo)]
    keys = np.ascontiguousarray(keys, dtype=np.int64)
    start = np.ascontiguousarray(start, dtype=np.uint64)
    length = np.ascontiguousarray(length, dtype=np.uint64)
    assert start.size == length.size
    out = np.zeros(start.size, dtype=np.uint64)
    info = _CopassInfo()
    rc = L.oc_copass_partition(keys.ctypes.data_as(C.c_void_p), start.ctypes.data_as(C.c_void_p),
                               length.ctypes.data_as(C.c_void_p), start.size, int(m),
                               out.ctypes.data_as(C.c_void_p), C.byref(info))
    if rc != 0:
        raise OracleError(rc)
    return out, info.t, info.iterations, info.last_step


def copass_block_sort(keys, vals, sizes, max_extract=None):
    """oc_copass_block_sort on copies of keys (int64) / vals (uint32); blocks of the given sizes lie one after the
    other.  Returns (keys, vals, sub_start, sub_len, stats dict)."""
    L = lib()
    L.oc_copass_block_sort.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_uint32, C.c_uint32, C.c_void_p,
                                       C.c_void_p, C.POINTER(_CopassStats)]
    keys = np.array(keys, dtype=np.int64)
    vals = np.array(vals, dtype=np.uint32)
    sizes = np.ascontiguousarray(sizes, dtype=np.uint64)
    assert keys.size == vals.size == int(sizes.sum())
    k = sizes.size
    sub_start, sub_len = np.zeros(k, dtype=np.uint64), np.zeros(k, dtype=np.uint64)
    st = _CopassStats()
    rc = L.oc_copass_block_sort(keys.ctypes.data_as(C.c_void_p), vals.ctypes.data_as(C.c_void_p),
                                sizes.ctypes.data_as(C.c_void_p), k, k if max_extract is None else int(max_extract),
                                sub_start.ctypes.data_as(C.c_void_p), sub_len.ctypes.data_as(C.c_void_p), C.byref(st))
    if rc != 0:
        raise OracleError(rc)
    return keys, vals, sub_start, sub_len, {f: getattr(st, f) for f, _ in _CopassStats._fields_}


NO_AUTAPSES, NO_MULTAPSES = 1, 2


def keyed_permutation(M: int, k: int, keys) -> int:
    """oc_keyed_permutation (reading A5)."""
    L = lib()
    L.oc_keyed_permutation.restype = C.c_uint32
    L.oc_keyed_permutation.argtypes = [C.c_uint32, C.c_uint32, C.POINTER(C.c_uint32)]
    arr = (C.c_uint32 * 4)(*[int(x) & 0xffffffff for x in keys])
    return int(L.oc_keyed_permutation(int(M), int(k), arr))
