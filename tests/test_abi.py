"""The C-ABI library builds for sm_100a on a machine without a GPU, loads, exports every symbol that
include/*.h declare, and refuses to run without a device (no CPU fallback).  CPU only."""
import ctypes
import re
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parent.parent


@pytest.fixture(scope="module")
def lib():
    from paper_2306_09855_b200 import build
    return ctypes.CDLL(str(build.build()))


def declared_symbols():
    """every function any header under include/ declares"""
    names = set()
    for h in sorted((ROOT / "include").glob("*.h")):
        text = re.sub(r"/\*.*?\*/", "", h.read_text(), flags=re.S)
        names |= set(re.findall(r"\b(nc_[a-z_0-9]+)\s*\(", text))
    return sorted(names)


def test_header_symbols_exported(lib):
    from paper_2306_09855_b200 import binding
    names = declared_symbols()
    assert len(names) >= 19
    for n in names:
        assert hasattr(lib, n), f"libnc.so does not export {n}"
    assert sorted(binding.SYMBOLS) == names, "binding.SYMBOLS out of step with include/*.h"


def test_struct_layouts_match_header():
    """sizeof of the ctypes mirrors = what a C compiler gives for include/nc.h (gcc, x86-64)."""
    import subprocess
    import tempfile
    from paper_2306_09855_b200 import binding as b
    src = '#include "nc.h"\n#include <stdio.h>\nint main(){printf("%zu %zu %zu %zu %zu %zu %zu %zu %zu %zu\\n",' \
          'sizeof(nc_config),sizeof(nc_rule_params),sizeof(nc_dist),sizeof(nc_syn_spec),sizeof(nc_range),' \
          'sizeof(nc_connections_view),sizeof(nc_index_view),sizeof(nc_timings),sizeof(nc_stats),sizeof(nc_allocator));return 0;}'
    with tempfile.TemporaryDirectory() as d:
        (Path(d) / "t.c").write_text(src)
        subprocess.run(["gcc", "-I", str(ROOT / "include"), "-o", f"{d}/t", f"{d}/t.c"], check=True)
        out = subprocess.run([f"{d}/t"], check=True, capture_output=True, text=True).stdout.split()
    want = [ctypes.sizeof(x) for x in (b.Config, b.RuleParams, b.Dist, b.SynSpec, b.Range, b.ConnectionsView,
                                       b.IndexView, b.Timings, b.Stats, b.Allocator)]
    assert [int(v) for v in out] == want


def test_constants_match_header():
    """the binding's status codes, NC_FLAG_* bits and rule flags are the header's values (compiled by gcc)."""
    import subprocess
    import tempfile
    from paper_2306_09855_b200 import binding as b
    pairs = [("NC_OK", b.OK), ("NC_ERR_INVALID_ARG", b.ERR_INVALID_ARG), ("NC_ERR_STATE", b.ERR_STATE),
             ("NC_ERR_CAPACITY", b.ERR_CAPACITY), ("NC_ERR_OOM", b.ERR_OOM), ("NC_ERR_CUDA", b.ERR_CUDA),
             ("NC_FLAG_TIMING", b.FLAG_TIMING), ("NC_FLAG_EXACT_FP64", b.FLAG_EXACT_FP64), ("NC_FLAG_SORT_PAIRS", b.FLAG_SORT_PAIRS),
             ("NC_FLAG_SORT_ONESWEEP", b.FLAG_SORT_ONESWEEP), ("NC_FLAG_ORGANISE_COPASS", b.FLAG_ORGANISE_COPASS),
             ("NC_FLAG_COPASS_SHIFT", b.FLAG_COPASS_SHIFT), ("NC_FLAG_SORT_BULK", b.FLAG_SORT_BULK),
             ("NC_FLAG_SORT_BUCKETS", b.FLAG_SORT_BUCKETS), ("NC_NO_AUTAPSES", b.NO_AUTAPSES), ("NC_NO_MULTAPSES", b.NO_MULTAPSES)]
    header = re.sub(r"/\*.*?\*/", "", (ROOT / "include" / "nc.h").read_text(), flags=re.S)
    declared = set(re.findall(r"\b(NC_FLAG_[A-Z_0-9]+)\s*=", header))
    assert declared == {n for n, _ in pairs if n.startswith("NC_FLAG_")}, "a flag of nc.h has no constant in binding.py"
    src = '#include "nc.h"\n#include <stdio.h>\nint main(){' + "".join(f'printf("%d\\n",(int){n});' for n, _ in pairs) + "return 0;}"
    with tempfile.TemporaryDirectory() as d:
        (Path(d) / "t.c").write_text(src)
        subprocess.run(["gcc", "-I", str(ROOT / "include"), "-o", f"{d}/t", f"{d}/t.c"], check=True)
        out = subprocess.run([f"{d}/t"], check=True, capture_output=True, text=True).stdout.split()
    assert [int(v) for v in out] == [v for _, v in pairs]


def test_no_cpu_fallback_without_gpu(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    from paper_2306_09855_b200 import binding as b
    cfg = b.Config()
    cfg.dt_ms = 0.1
    cfg.device = -1
    h = ctypes.c_void_p()
    L = b.load_library()
    assert L.nc_create(ctypes.byref(cfg), ctypes.byref(h)) == b.ERR_CUDA and not h.value
    with pytest.raises(RuntimeError):
        b.NC()


def test_invalid_config_rejected(lib):
    from paper_2306_09855_b200 import binding as b
    L = b.load_library()
    cfg = b.Config()
    cfg.dt_ms = 0.0
    h = ctypes.c_void_p()
    assert L.nc_create(ctypes.byref(cfg), ctypes.byref(h)) == b.ERR_INVALID_ARG
    assert L.nc_create(None, ctypes.byref(h)) == b.ERR_INVALID_ARG
