"""The CUDA path against library routines the product never links ("GPU-side independent check"):
cuRAND's own Philox4x32-10 for the device RNG, cub::DeviceRadixSort::SortPairs -- the sort underneath the paper's
block-sort -- for the organised order.  tests/cuda/comparators.cu is test-only code built here."""
import ctypes as C
import subprocess
from pathlib import Path

import numpy as np
import pytest

from paper_2306_09855_b200 import workloads as WL

pytestmark = pytest.mark.gpu
HERE = Path(__file__).resolve().parent / "cuda"


@pytest.fixture(scope="module")
def nc_mod():
    from paper_2306_09855_b200 import binding, build
    build.build()
    return binding


@pytest.fixture(scope="module")
def cmp_lib():
    src, lib = HERE / "comparators.cu", HERE / "libcmp.so"
    if not lib.exists() or lib.stat().st_mtime < src.stat().st_mtime:
        subprocess.run(["/usr/local/cuda/bin/nvcc", "-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a",
                        "-Xcompiler", "-fPIC", "-shared", "-o", str(lib), str(src)], check=True)
    L = C.CDLL(str(lib))
    L.cmp_curand_philox.argtypes = [C.c_uint32, C.c_void_p, C.c_void_p, C.c_void_p]
    L.cmp_cub_sort_pairs.argtypes = [C.c_uint32, C.c_void_p, C.c_void_p, C.c_int, C.c_int, C.POINTER(C.c_float),
                                     C.POINTER(C.c_uint64)]
    return L


def test_device_philox_equals_curand_round_function(nc_mod, cmp_lib):
    rng = np.random.default_rng(5)
    n = 100_000
    ctr = rng.integers(0, 2**32, size=(n, 4), dtype=np.uint64).astype(np.uint32)
    key = rng.integers(0, 2**32, size=(n, 2), dtype=np.uint64).astype(np.uint32)
    ref = np.empty_like(ctr)
    assert cmp_lib.cmp_curand_philox(n, ctr.ctypes.data, key.ctypes.data, ref.ctypes.data) == 0
    g = nc_mod.NC()
    assert np.array_equal(g.selftest_philox(ctr, key), ref)
    g.close()


def _cub_perm(cmp_lib, keys_host, key_bits):
    import torch
    d_keys = torch.from_numpy(keys_host.astype(np.int64)).to(torch.int64).cuda().to(torch.int32)  # bit pattern of u32
    d_perm = torch.empty(keys_host.size, dtype=torch.int32, device="cuda")
    torch.cuda.synchronize()
    ms, tmp = C.c_float(), C.c_uint64()
    rc = cmp_lib.cmp_cub_sort_pairs(keys_host.size, d_keys.data_ptr(), d_perm.data_ptr(), 0, key_bits, C.byref(ms), C.byref(tmp))
    assert rc == 0
    return d_perm.cpu().numpy().view(np.uint32), ms.value, tmp.value


@pytest.mark.parametrize("flags_name", ["default", "copass"])
def test_organised_order_equals_cub_sort_pairs(nc_mod, cmp_lib, flags_name):
    net = WL.config2_microcircuit(scale=0.1)
    flags = nc_mod.FLAG_ORGANISE_COPASS if flags_name == "copass" else 0
    g = nc_mod.NC(dt_ms=net.dt_ms, flags=flags, block_size=1 << 18)
    WL.run(net, g, finalize=False)
    u = g.read_connections(sorted=False, fields=("source", "delay"))
    g.finalize()
    st = g.stats()
    keys = (u["source"].astype(np.uint64) << np.uint64(st["delay_bits"])) | u["delay"].astype(np.uint64)
    assert int(keys.max()) < 2**32
    perm, _, _ = _cub_perm(cmp_lib, keys.astype(np.uint32), st["key_bits"])
    assert np.array_equal(g.read_connections(sorted=True, fields=("perm",))["perm"], perm)
    g.close()


def test_cub_sort_pairs_context_timing_full_size(nc_mod, cmp_lib):
    """Context number: cub::DeviceRadixSort::SortPairs on the (key, position) pairs of configs[2] at full
    size on this GPU -- the paper's underlying sort; it orders positions only, target and weight still have to be
    gathered.  The permutation must equal the library's."""
    net = WL.config2_microcircuit()
    g = nc_mod.NC(dt_ms=net.dt_ms)
    WL.run(net, g, finalize=False)
    u = g.read_connections(sorted=False, fields=("source", "delay"))
    g.finalize()
    st = g.stats()
    keys = ((u["source"].astype(np.uint64) << np.uint64(st["delay_bits"])) | u["delay"].astype(np.uint64)).astype(np.uint32)
    del u
    perm, ms, tmp = _cub_perm(cmp_lib, keys, st["key_bits"])
    print(f"cub::DeviceRadixSort::SortPairs, {keys.size} pairs, {st['key_bits']} key bits: {ms:.3f} ms, "
          f"{tmp / 1e6:.1f} MB temporary storage")
    assert np.array_equal(g.read_connections(sorted=True, fields=("perm",))["perm"], perm)
    g.close()
