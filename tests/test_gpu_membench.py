"""Runs the test-only microbenchmarks of tests/cuda/membench.cu on the device and keeps their tables
(gpurun_out/membench.txt).  They are the measurements behind two bounds DESIGN.md states:
  * the ceiling of a digit pass's write pattern (runs of 16-byte records that start inside a 32-byte sector) against an
    aligned copy -- section 6.3;
  * the issue cost of the Philox multiplies -- section 6.1;
  * what keeping a pass's intermediate array in the L2 can gain (section `ring`) -- section 6.3, bucket-first organisation.
Assertions are deliberately loose (they check that the tables exist and say what DESIGN.md relies on, not absolute rates)."""
import re
import subprocess
from pathlib import Path

import pytest

pytestmark = pytest.mark.gpu
HERE = Path(__file__).resolve().parent / "cuda"
OUT = Path(__file__).resolve().parent.parent / "gpurun_out"


@pytest.fixture(scope="module")
def membench():
    src, exe = HERE / "membench.cu", HERE / "membench"
    if not exe.exists() or exe.stat().st_mtime < src.stat().st_mtime:
        subprocess.run(["/usr/local/cuda/bin/nvcc", "-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a",
                        "-o", str(exe), str(src)], check=True)
    return exe


def _run(exe, what):
    r = subprocess.run([str(exe), what], capture_output=True, text=True, timeout=600)
    assert r.returncode == 0, r.stdout + r.stderr
    OUT.mkdir(exist_ok=True)
    with open(OUT / "membench.txt", "a") as f:
        f.write(r.stdout)
    return r.stdout


def _rows(text):
    return [[c.strip() for c in line.strip("|").split("|")] for line in text.splitlines()
            if line.startswith("|") and not line.startswith("|---") and re.match(r"\|\s*[\d.]", line)]


def test_shared_atomics_of_one_warp_instruction_are_served_in_lane_order(membench):
    out = _run(membench, "atomorder")
    assert "atomorder violations total: 0" in out, out


def test_write_pattern_ceiling(membench):
    out = _run(membench, "pattern")
    rows = {(int(r[0]), int(r[1]), int(r[2]), int(r[3])): float(r[5]) for r in _rows(out)}
    aligned, sector_split = rows[(256, 256, 0, 1)], rows[(256, 256, 16, 1)]
    # pieces that start inside a sector cost bandwidth: this is the pattern a scatter pass of 16-byte records writes
    assert sector_split < 0.9 * aligned, out
    assert rows[(256, 256, 32, 1)] > sector_split, out


def test_l2_resident_intermediate(membench):
    """Two passes with the intermediate array kept in the L2 group by group against two whole-array passes (DESIGN.md 6.3,
    bucket-first organisation): the memory system alone gains from it."""
    out = _run(membench, "ring")
    rows = [l for l in out.splitlines() if l.startswith("|") and ("ring" in l or "full" in l) and not l.startswith("| group")]
    ms = lambda l: float(l.strip("|").split("|")[-2])
    whole = ms([l for l in rows if l.startswith("| whole array")][0])
    best_ring = min(ms(l) for l in rows if "| ring |" in l)
    assert best_ring < 0.85 * whole, out


def test_bulk_copy_path(membench):
    out = _run(membench, "bulk")
    assert len(_rows(out)) >= 6, out


def test_pipe_rates(membench):
    out = _run(membench, "pipes")
    wide = [r for r in out.splitlines() if r.startswith("| IMAD.WIDE")]
    assert wide, out
    cyc = float(wide[0].strip("|").split("|")[-1])
    assert 1.0 < cyc < 16.0, out


def test_scattered_reduction_ceiling(membench):
    out = _run(membench, "red")
    assert len(_rows(out)) == 4, out
