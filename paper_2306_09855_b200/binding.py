"""Thin ctypes binding over libnc.so (C ABI: include/nc.h) -- argument marshalling only.

Every step of the path (rule expansion, draws, append, sort, index) runs in the CUDA kernels of the
library.  PyTorch is used for two things: device memory (the library's nc_allocator callbacks are backed by
torch's caching allocator) and the CUDA stream the work is enqueued on.  There is no CPU fallback: without
the built library or without a GPU, creating a context raises.
"""
from __future__ import annotations

import ctypes as C
import weakref
import math
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
LIB_PATH = _HERE / "libnc.so"

OK, ERR_INVALID_ARG, ERR_STATE, ERR_CAPACITY, ERR_OOM, ERR_CUDA = 0, -1, -2, -3, -4, -5
ONE_TO_ONE, ALL_TO_ALL, FIXED_INDEGREE, FIXED_OUTDEGREE, FIXED_TOTAL_NUMBER, PAIRWISE_BERNOULLI = range(6)
FLAG_TIMING, FLAG_EXACT_FP64, FLAG_SORT_PAIRS, FLAG_SORT_ONESWEEP, FLAG_ORGANISE_COPASS, FLAG_COPASS_SHIFT = 1, 2, 4, 8, 16, 32
FLAG_SORT_BULK = 64
FLAG_SORT_BUCKETS = 128
NO_AUTAPSES, NO_MULTAPSES = 1, 2  # nc_set_rule_flags
PHASES = ("generate", "histogram", "sort", "permute", "index", "degree", "copass")

# every symbol include/nc.h declares (checked by tests/test_abi.py against the header and the library)
SYMBOLS = (
    "nc_create", "nc_destroy", "nc_last_error", "nc_synchronize", "nc_create_population", "nc_connect",
    "nc_finalize", "nc_num_connections", "nc_num_nodes", "nc_get_connections", "nc_get_index",
    "nc_degree_histogram", "nc_get_stats", "nc_get_timings", "nc_read_connections", "nc_read_index",
    "nc_read_degree_histogram", "nc_selftest_philox", "nc_selftest_fastpath", "nc_selftest_guard",
    "nc_connect_nodes", "nc_connect_values", "nc_set_connection_attributes", "nc_read_connection_attributes",
    "nc_set_rule_flags", "nc_set_shard",
    # include/nc_delivery.h
    "nc_delivery_create", "nc_delivery_destroy", "nc_delivery_step", "nc_delivery_read_spike_array",
    "nc_delivery_counts", "nc_delivery_num_ports", "nc_delivery_run",
    # include/nc_copass.h
    "nc_copass_partition", "nc_get_copass_stats",
    # include/nc_static.h
    "nc_index_static",
)

ALLOC_FN = C.CFUNCTYPE(C.c_void_p, C.c_void_p, C.c_size_t)
FREE_FN = C.CFUNCTYPE(None, C.c_void_p, C.c_void_p)


class Allocator(C.Structure):
    _fields_ = [("alloc", ALLOC_FN), ("free", FREE_FN), ("user", C.c_void_p)]


class Config(C.Structure):
    _fields_ = [("block_size", C.c_uint64), ("dt_ms", C.c_double), ("mem", Allocator),
                ("cuda_stream", C.c_void_p), ("device", C.c_int32), ("flags", C.c_uint32)]


class RuleParams(C.Structure):
    _fields_ = [("degree_or_total", C.c_uint64), ("p", C.c_double)]


class Dist(C.Structure):
    _fields_ = [("mean", C.c_double), ("sd", C.c_double), ("lo", C.c_double), ("hi", C.c_double)]


class SynSpec(C.Structure):
    _fields_ = [("weight", Dist), ("delay_ms", Dist)]


class Range(C.Structure):
    _fields_ = [("first", C.c_uint32), ("count", C.c_uint32)]


class ConnectionsView(C.Structure):
    _fields_ = [("source", C.c_void_p), ("target", C.c_void_p), ("weight", C.c_void_p), ("delay", C.c_void_p),
                ("perm", C.c_void_p), ("n", C.c_uint64), ("block_size", C.c_uint64), ("n_blocks", C.c_uint64),
                ("blocks", C.POINTER(C.c_void_p)), ("off_source", C.c_uint64), ("off_target", C.c_uint64),
                ("off_weight", C.c_uint64), ("off_delay", C.c_uint64), ("off_perm", C.c_uint64)]


class IndexView(C.Structure):
    _fields_ = [("src_offsets", C.c_void_p), ("group_count", C.c_void_p), ("group_ptr", C.c_void_p),
                ("group_start", C.c_void_p), ("group_delay", C.c_void_p), ("n_nodes", C.c_uint32),
                ("total_groups", C.c_uint32)]


class Timings(C.Structure):
    _fields_ = [("ms", C.c_double * 7), ("launches", C.c_uint32 * 7), ("sort_pass_ms", C.c_double),
                ("sort_passes", C.c_uint32)]


class Stats(C.Structure):
    _fields_ = [("kernel_launches", C.c_uint64), ("bytes_in_use", C.c_uint64), ("bytes_peak", C.c_uint64),
                ("n_blocks", C.c_uint64), ("n_projections", C.c_uint32), ("key_bits", C.c_uint32),
                ("sort_passes", C.c_uint32), ("delay_bits", C.c_uint32)]


class CopassInfo(C.Structure):
    _fields_ = [("t", C.c_uint32), ("iterations", C.c_uint32), ("last_step", C.c_int32)]


class CopassStats(C.Structure):
    _fields_ = [("partitions", C.c_uint32), ("iterations", C.c_uint32), ("last_step_1", C.c_uint32),
                ("last_step_2", C.c_uint32), ("n_blocks", C.c_uint64), ("aux_bytes", C.c_uint64),
                ("records_moved", C.c_uint64)]


_lib = None


def load_library():
    """dlopen libnc.so and declare the argument types of every entry point.  Raises if it is not built."""
    global _lib
    if _lib is not None:
        return _lib
    import os
    path = Path(os.environ.get("NC_LIB_PATH", str(LIB_PATH)))  # development override: another build of the same ABI
    if not path.exists():
        raise RuntimeError(f"{path} is not built: run `python -m paper_2306_09855_b200.build` "
                           "(there is no CPU fallback)")
    L = C.CDLL(str(path))
    P, vp = C.POINTER, C.c_void_p
    L.nc_create.argtypes = [P(Config), P(vp)]
    L.nc_destroy.argtypes = [vp]
    L.nc_last_error.argtypes = [vp]
    L.nc_last_error.restype = C.c_char_p
    L.nc_synchronize.argtypes = [vp]
    L.nc_create_population.argtypes = [vp, C.c_uint32, P(C.c_uint32)]
    L.nc_connect.argtypes = [vp, Range, Range, C.c_int, P(RuleParams), P(SynSpec), C.c_uint64]
    L.nc_finalize.argtypes = [vp]
    L.nc_num_connections.argtypes = [vp, P(C.c_uint64)]
    L.nc_num_nodes.argtypes = [vp, P(C.c_uint32)]
    L.nc_get_connections.argtypes = [vp, C.c_int, P(ConnectionsView)]
    L.nc_get_index.argtypes = [vp, P(IndexView)]
    L.nc_degree_histogram.argtypes = [vp, C.c_int, P(vp), P(C.c_uint32)]
    L.nc_get_stats.argtypes = [vp, P(Stats)]
    L.nc_get_timings.argtypes = [vp, P(Timings)]
    L.nc_read_connections.argtypes = [vp, C.c_int, C.c_uint64, C.c_uint64, vp, vp, vp, vp, vp]
    L.nc_read_index.argtypes = [vp, vp, vp, vp, vp, vp]
    L.nc_read_degree_histogram.argtypes = [vp, C.c_int, vp, P(C.c_uint32)]
    L.nc_selftest_philox.argtypes = [vp, C.c_uint32, vp, vp, vp]
    L.nc_selftest_fastpath.argtypes = [vp, P(C.c_double)]
    L.nc_selftest_guard.argtypes = [vp, C.c_int, P(C.c_uint64)]
    L.nc_connect_nodes.argtypes = [vp, vp, C.c_uint32, Range, vp, C.c_uint32, Range, C.c_int, vp, vp, C.c_uint64]
    L.nc_copass_partition.argtypes = [vp, vp, C.c_uint64, vp, vp, C.c_uint32, C.c_uint32, vp, P(CopassInfo)]
    L.nc_get_copass_stats.argtypes = [vp, P(CopassStats)]
    L.nc_connect_values.argtypes = [vp, vp, C.c_uint32, Range, vp, C.c_uint32, Range, C.c_int, vp, vp, C.c_uint64, vp, vp,
                                    C.c_uint64]
    L.nc_set_connection_attributes.argtypes = [vp, C.c_uint8, C.c_uint8]
    L.nc_read_connection_attributes.argtypes = [vp, C.c_int, C.c_uint64, C.c_uint64, vp, vp]
    L.nc_delivery_create.argtypes = [vp, C.c_uint32, P(vp)]
    L.nc_delivery_destroy.argtypes = [vp]
    L.nc_delivery_num_ports.argtypes = [vp, P(C.c_uint32)]
    L.nc_delivery_run.argtypes = [vp, C.c_uint32, vp, vp, vp, vp]
    L.nc_delivery_step.argtypes = [vp, vp, vp, C.c_uint32, vp]
    L.nc_delivery_read_spike_array.argtypes = [vp, vp, vp, C.c_uint32, P(C.c_uint32)]
    L.nc_delivery_counts.argtypes = [vp, P(C.c_uint64), P(C.c_uint64), P(C.c_uint64), P(C.c_uint64)]
    L.nc_index_static.argtypes = [vp, vp, C.c_uint64, C.c_uint32, vp, vp, vp, vp, vp, C.c_uint64, vp, vp, vp, C.c_char_p,
                                  C.c_size_t]
    for name in SYMBOLS:
        if name != "nc_last_error":
            getattr(L, name).restype = C.c_int
    _lib = L
    return L


class NCError(RuntimeError):
    def __init__(self, code, msg=""):
        super().__init__(f"nc error {code}: {msg}")
        self.code = code


def _ptr(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


INDEX_STATIC_MAX_CONNECTIONS = 1 << 30  # NC_INDEX_STATIC_MAX_CONNECTIONS (include/nc_static.h)
INDEX_STATIC_LOOKBACK, INDEX_STATIC_GROUPS = 1, 2


def index_static(d_source, d_delay, n, n_nodes, d_src_offsets, d_group_ptr, d_group_count, d_group_start, d_group_delay,
                 group_capacity, d_total_groups, d_error, stream=None):
    """nc_index_static (include/nc_static.h): the group index over organised connections, built without any device
    allocation -- for callers that cannot allocate where they need it (a loop with a latency budget, a process whose own
    pool already owns the whole card).  The scratch is an array inside the library image, shared by all calls on a
    device: calls that overlap on the GPU race.  Every d_* argument is a raw device address (int; tensor.data_ptr()) or
    None where the header allows NULL; the caller owns those buffers.  The work is enqueued on `stream` (a torch stream;
    default: the current one) of the current device and not waited for.  Raises NCError with the library's message,
    e.g. ERR_CAPACITY for n > INDEX_STATIC_MAX_CONNECTIONS."""
    import torch
    L = load_library()
    s = stream if stream is not None else torch.cuda.current_stream()
    msg = C.create_string_buffer(512)
    rc = L.nc_index_static(d_source, d_delay, int(n), int(n_nodes), d_src_offsets, d_group_ptr, d_group_count, d_group_start,
                           d_group_delay, int(group_capacity), d_total_groups, d_error, s.cuda_stream, msg, 512)
    if rc != 0:
        raise NCError(rc, msg.value.decode())


def _host_buffer(n, dtype):
    """Host array for a device -> host read: page-locked (torch's caching host allocator), so the copy runs at PCIe
    speed instead of being staged through a bounce buffer; plain numpy memory if pinning is not possible."""
    dtype = np.dtype(dtype)
    if int(n) * dtype.itemsize > (256 << 20):  # do not page-lock gigabytes
        return np.empty(int(n), dtype=dtype)
    try:
        import torch
        t = torch.empty(int(n) * dtype.itemsize, dtype=torch.uint8, pin_memory=True)
        return t.numpy().view(dtype)  # the view keeps the tensor alive
    except Exception:
        return np.empty(int(n), dtype=dtype)


class TorchAllocator:
    """nc_allocator backed by torch's caching allocator on the current device/stream."""

    def __init__(self):
        import torch
        self._torch = torch
        self._held = {}
        self.alloc_cb = ALLOC_FN(self._alloc)
        self.free_cb = FREE_FN(self._free)

    def _alloc(self, _user, nbytes):
        try:
            t = self._torch.empty(int(nbytes), dtype=self._torch.uint8, device="cuda")
        except Exception:  # torch.cuda.OutOfMemoryError and friends -> NULL -> NC_ERR_OOM
            return None
        p = t.data_ptr()
        self._held[p] = t
        return p

    def _free(self, _user, p):
        self._held.pop(p, None)

    def struct(self):
        return Allocator(self.alloc_cb, self.free_cb, None)


class NC:
    """One construction context.  Method names and order follow the C ABI one to one."""

    def __init__(self, dt_ms: float = 0.1, block_size: int = 0, flags: int = 0, use_torch_allocator: bool = True,
                 stream=None):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("no CUDA device: the construction path only exists as CUDA kernels (no CPU fallback)")
        self._L = load_library()
        self._alloc = TorchAllocator() if use_torch_allocator else None
        cfg = Config()
        cfg.block_size = int(block_size)
        cfg.dt_ms = float(dt_ms)
        if self._alloc is not None:
            cfg.mem = self._alloc.struct()
        s = stream if stream is not None else torch.cuda.current_stream()
        self._stream = s
        cfg.cuda_stream = s.cuda_stream
        cfg.device = torch.cuda.current_device()
        cfg.flags = int(flags)
        self._h = C.c_void_p()
        self._deliveries = weakref.WeakSet()  # closed before the context: they allocate from it (nc_delivery.h)
        rc = self._L.nc_create(C.byref(cfg), C.byref(self._h))
        if rc != 0:
            raise NCError(rc, "nc_create failed")

    # -- plumbing --
    def _check(self, rc):
        if rc != 0:
            raise NCError(rc, (self._L.nc_last_error(self._h) or b"").decode())

    def close(self):
        if getattr(self, "_h", None):
            for d in list(getattr(self, "_deliveries", ())):
                d.close()
            rc = self._L.nc_destroy(self._h)
            self._h = C.c_void_p()
            if rc != 0:  # NC_GUARD=1: a guard zone around one of the library's buffers was overwritten
                raise NCError(rc, "nc_destroy: guard zone violation (see stderr)")

    def guard_violations(self) -> int:
        self._L.nc_internal_guard_violations.restype = C.c_uint64
        self._L.nc_internal_guard_violations.argtypes = [C.c_void_p]
        return int(self._L.nc_internal_guard_violations(self._h))

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()

    # -- the ABI --
    def synchronize(self):
        self._check(self._L.nc_synchronize(self._h))

    def create_population(self, n: int) -> int:
        first = C.c_uint32()
        self._check(self._L.nc_create_population(self._h, int(n), C.byref(first)))
        return first.value

    def connect_rc(self, src, tgt, rule, degree_or_total=0, p=0.0, weight=(1.0, 0.0, -math.inf, math.inf),
                   delay_ms=(1.0, 0.0, -math.inf, math.inf), seed=0, weights=None, delays=None) -> int:
        """weights / delays: per-connection value arrays on the host (nc_connect_values); None = follow the
        distributions."""
        rp = RuleParams(int(degree_or_total), float(p))
        sp = SynSpec(Dist(*map(float, weight)), Dist(*map(float, delay_ms)))
        if weights is not None or delays is not None:
            sa = None if isinstance(src, tuple) else np.ascontiguousarray(src, dtype=np.uint32)
            ta = None if isinstance(tgt, tuple) else np.ascontiguousarray(tgt, dtype=np.uint32)
            wa = None if weights is None else np.ascontiguousarray(weights, dtype=np.float32)
            da = None if delays is None else np.ascontiguousarray(delays, dtype=np.float64)
            return int(self._L.nc_connect_values(self._h, _ptr(sa), 0 if sa is None else sa.size,
                                                 Range(0, 0) if sa is not None else Range(*src), _ptr(ta),
                                                 0 if ta is None else ta.size,
                                                 Range(0, 0) if ta is not None else Range(*tgt), int(rule), C.byref(rp),
                                                 C.byref(sp), int(seed), _ptr(wa), _ptr(da),
                                                 (wa if wa is not None else da).size))
        if isinstance(src, tuple) and isinstance(tgt, tuple):
            return int(self._L.nc_connect(self._h, Range(*src), Range(*tgt), int(rule), C.byref(rp), C.byref(sp), int(seed)))
        # a side that is not a (first, count) tuple is an explicit host array of node ids (nc_connect_nodes)
        sa = None if isinstance(src, tuple) else np.ascontiguousarray(src, dtype=np.uint32)
        ta = None if isinstance(tgt, tuple) else np.ascontiguousarray(tgt, dtype=np.uint32)
        return int(self._L.nc_connect_nodes(self._h, _ptr(sa), 0 if sa is None else sa.size,
                                            Range(0, 0) if sa is not None else Range(*src), _ptr(ta),
                                            0 if ta is None else ta.size, Range(0, 0) if ta is not None else Range(*tgt),
                                            int(rule), C.byref(rp), C.byref(sp), int(seed)))

    def connect(self, *a, **k):
        self._check(self.connect_rc(*a, **k))

    def set_shard(self, first: int, count: int):
        self._L.nc_set_shard.argtypes = [C.c_void_p, C.c_uint32, C.c_uint32]
        self._check(self._L.nc_set_shard(self._h, int(first), int(count)))

    def set_rule_flags(self, flags: int):
        self._L.nc_set_rule_flags.argtypes = [C.c_void_p, C.c_uint32]
        self._check(self._L.nc_set_rule_flags(self._h, int(flags)))

    def set_connection_attributes(self, port: int, syn_group: int = 0):
        self._check(self._L.nc_set_connection_attributes(self._h, int(port), int(syn_group)))

    def read_connection_attributes(self, sorted: bool = False, first: int = 0, count: int | None = None):
        if count is None:
            count = self.num_connections() - first
        port, group = np.zeros(int(count), np.uint8), np.zeros(int(count), np.uint8)
        self._check(self._L.nc_read_connection_attributes(self._h, 1 if sorted else 0, int(first), int(count), _ptr(port),
                                                          _ptr(group)))
        return port, group

    def finalize(self):
        self._check(self._L.nc_finalize(self._h))

    def num_connections(self) -> int:
        n = C.c_uint64()
        self._check(self._L.nc_num_connections(self._h, C.byref(n)))
        return n.value

    def num_nodes(self) -> int:
        n = C.c_uint32()
        self._check(self._L.nc_num_nodes(self._h, C.byref(n)))
        return n.value

    def get_connections(self, sorted: bool = False) -> ConnectionsView:
        v = ConnectionsView()
        self._check(self._L.nc_get_connections(self._h, 1 if sorted else 0, C.byref(v)))
        return v

    def get_index(self) -> IndexView:
        v = IndexView()
        self._check(self._L.nc_get_index(self._h, C.byref(v)))
        return v

    def stats(self) -> dict:
        s = Stats()
        self._check(self._L.nc_get_stats(self._h, C.byref(s)))
        return {f: getattr(s, f) for f, _ in Stats._fields_}

    def timings(self) -> dict:
        t = Timings()
        self._check(self._L.nc_get_timings(self._h, C.byref(t)))
        out = {f"{name}_ms": t.ms[i] for i, name in enumerate(PHASES)}
        out["sort_pass_ms"] = t.sort_pass_ms
        out["sort_passes"] = t.sort_passes
        return out

    # -- host-buffer reads --
    def read_connections(self, sorted: bool = False, first: int = 0, count: int | None = None,
                         fields=("source", "target", "weight", "delay", "perm")) -> dict:
        n = self.num_connections()
        if count is None:
            count = n - first
        out = {"n": int(count)}
        bufs = {"source": np.uint32, "target": np.uint32, "weight": np.float32, "delay": np.uint16, "perm": np.uint32}
        arr = {k: (_host_buffer(count, dt) if (k in fields and (k != "perm" or sorted)) else None)
               for k, dt in bufs.items()}
        self._check(self._L.nc_read_connections(self._h, 1 if sorted else 0, int(first), int(count), _ptr(arr["source"]),
                                                _ptr(arr["target"]), _ptr(arr["weight"]), _ptr(arr["delay"]),
                                                _ptr(arr["perm"])))
        out.update({k: v for k, v in arr.items() if v is not None})
        return out

    def read_index(self) -> dict:
        v = self.get_index()
        N, G = v.n_nodes, v.total_groups
        a = {"src_offsets": _host_buffer(N + 1, np.uint32), "group_count": _host_buffer(N, np.uint32),
             "group_ptr": _host_buffer(N + 1, np.uint32), "group_start": _host_buffer(G, np.uint32),
             "group_delay": _host_buffer(G, np.uint16)}
        self._check(self._L.nc_read_index(self._h, _ptr(a["src_offsets"]), _ptr(a["group_count"]), _ptr(a["group_ptr"]),
                                          _ptr(a["group_start"]), _ptr(a["group_delay"])))
        a["n_nodes"], a["total_groups"] = int(N), int(G)
        return a

    def read_degree_histogram(self, kind: int):
        deg = np.empty(self.num_nodes(), np.uint32)
        mx = C.c_uint32()
        self._check(self._L.nc_read_degree_histogram(self._h, int(kind), _ptr(deg), C.byref(mx)))
        return deg, mx.value

    # -- COPASS block-sort (include/nc_copass.h) --
    def copass_partition(self, keys, start, length, m):
        """nc_copass_partition on host arrays: returns (m_i uint32[k], t, iterations, last_step)."""
        keys = np.ascontiguousarray(keys, dtype=np.uint32)
        start = np.ascontiguousarray(start, dtype=np.uint32)
        length = np.ascontiguousarray(length, dtype=np.uint32)
        out = np.zeros(start.size, dtype=np.uint32)
        info = CopassInfo()
        self._check(self._L.nc_copass_partition(self._h, _ptr(keys), keys.size, _ptr(start), _ptr(length), start.size,
                                                int(m), _ptr(out), C.byref(info)))
        return out, info.t, info.iterations, info.last_step

    def copass_stats(self) -> dict:
        s = CopassStats()
        self._check(self._L.nc_get_copass_stats(self._h, C.byref(s)))
        return {f: getattr(s, f) for f, _ in CopassStats._fields_}

    # -- device self-tests --
    def selftest_philox(self, ctr: np.ndarray, key: np.ndarray) -> np.ndarray:
        ctr = np.ascontiguousarray(ctr, dtype=np.uint32).reshape(-1, 4)
        key = np.ascontiguousarray(key, dtype=np.uint32).reshape(-1, 2)
        out = np.empty_like(ctr)
        self._check(self._L.nc_selftest_philox(self._h, ctr.shape[0], _ptr(ctr), _ptr(key), _ptr(out)))
        return out

    def selftest_guard(self, offset: int) -> int:
        v = C.c_uint64()
        self._check(self._L.nc_selftest_guard(self._h, int(offset), C.byref(v)))
        return v.value

    def selftest_fastpath(self):
        out = (C.c_double * 4)()
        self._check(self._L.nc_selftest_fastpath(self._h, out))
        return tuple(out)


class Delivery:
    """Spike delivery over a finalized NC context (include/nc_delivery.h).  Arguments of step() are
    torch CUDA tensors (uint32 / int32 node ids and multiplicities, float32 input): device memory only, every step
    of the path runs in the library's kernels."""

    def __init__(self, nc: NC, capacity: int):
        self._nc, self._L = nc, nc._L  # the context must outlive this object
        self._h = C.c_void_p()
        nc._check(self._L.nc_delivery_create(nc._h, int(capacity), C.byref(self._h)))
        self.capacity = int(capacity)
        n_ports = C.c_uint32()
        nc._check(self._L.nc_delivery_num_ports(self._h, C.byref(n_ports)))
        self.n_ports = n_ports.value
        nc._deliveries.add(self)

    def step(self, nodes, mult, input_f32, n_new=None):
        n = int(nodes.numel()) if n_new is None else int(n_new)
        assert input_f32.is_cuda and input_f32.element_size() == 4 and input_f32.numel() == self._nc.num_nodes() * self.n_ports
        assert nodes.is_cuda and nodes.element_size() == 4 and (mult is None or (mult.is_cuda and mult.element_size() == 4))
        self._nc._check(self._L.nc_delivery_step(self._h, nodes.data_ptr() if n else None,
                                                 mult.data_ptr() if (mult is not None and n) else None, n,
                                                 input_f32.data_ptr()))

    def run(self, nodes, mult, offsets, input_f32):
        """nc_delivery_run: len(offsets) - 1 steps over a raster resident on the device (nodes / mult: CUDA tensors;
        offsets: host integers, step k emits nodes[offsets[k]:offsets[k+1]])."""
        offs = np.ascontiguousarray(offsets, dtype=np.uint64)
        assert input_f32.is_cuda and input_f32.numel() == self._nc.num_nodes() * self.n_ports
        self._nc._check(self._L.nc_delivery_run(self._h, offs.size - 1, nodes.data_ptr(),
                                                None if mult is None else mult.data_ptr(), _ptr(offs),
                                                input_f32.data_ptr()))

    def read_spike_array(self):
        n = C.c_uint32()
        g, m = _host_buffer(self.capacity, np.uint32), _host_buffer(self.capacity, np.uint32)
        self._nc._check(self._L.nc_delivery_read_spike_array(self._h, _ptr(g), _ptr(m), self.capacity, C.byref(n)))
        return g[:n.value].copy(), m[:n.value].copy()

    def counts(self) -> dict:
        v = [C.c_uint64() for _ in range(4)]
        self._nc._check(self._L.nc_delivery_counts(self._h, *[C.byref(x) for x in v]))
        return dict(zip(("buffered", "events", "dropped", "bad_nodes"), (x.value for x in v)))

    def close(self):
        if getattr(self, "_h", None):
            self._L.nc_delivery_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
