"""compute-sanitizer is closed on the GPU pool these tests run on (profiles/r02_sanitizer.md), so the library carries
its own bounds check: NC_GUARD=1 puts every device buffer between two guard zones that are compared when the buffer is
released (include/nc.h, nc_selftest_guard).  Here: the check fires on a deliberate one-byte overrun on either side, and
the small cases of tests/sanitizer_cases.py -- every organisation variant and both delivery forms -- leave all guards
intact (a violation makes nc_destroy return NC_ERR_STATE, which NC.close() raises)."""
import os
import subprocess
import sys
from pathlib import Path

import pytest

pytestmark = pytest.mark.gpu
ROOT = Path(__file__).resolve().parent.parent


def test_guard_zones_catch_a_one_byte_overrun():
    from paper_2306_09855_b200 import binding, build
    build.build()
    os.environ["NC_GUARD"] = "1"
    try:
        g = binding.NC()
        assert g.selftest_guard(0) == 0
        assert g.selftest_guard(1) == 1
        assert g.selftest_guard(-1) == 1
        assert g.guard_violations() == 0
        g.close()
    finally:
        os.environ.pop("NC_GUARD")
    g = binding.NC()
    with pytest.raises(binding.NCError):
        g.selftest_guard(1)  # guards are off without NC_GUARD
    g.close()


def test_small_cases_of_every_variant_leave_the_guard_zones_intact():
    env = dict(os.environ, NC_GUARD="1")
    r = subprocess.run([sys.executable, str(ROOT / "tests" / "sanitizer_cases.py")], env=env, capture_output=True, text=True,
                       timeout=900)
    assert r.returncode == 0, r.stdout[-3000:] + r.stderr[-3000:]
    assert "sanitizer cases OK" in r.stdout and "libnc guard" not in r.stderr, r.stderr[-3000:]
