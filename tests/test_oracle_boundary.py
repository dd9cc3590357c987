"""Pins for the oracle's `boundary` flag (reading D8; PAPER.md:117 for the delay rule).

The flag is the oracle's statement of WHICH synapses may differ by one delay step on the GPU: those whose
pre-rounding value x = d_ms * inv_dt lies within 1e-9 of k + 1/2, and those whose d_ms is within 1e-12 relative
of a clip bound without being equal to it.  The GPU parity tests lean on it (tests/parity_util.py), so a band that
is too wide (1e-3 instead of 1e-9), or a clip test that also fires on exact clamps, would silently widen the GPU
tolerance.  Every expected value below is fixed by the definition D8 and IEEE arithmetic on constants chosen by
hand, not by the oracle.  CPU only."""
import math

import numpy as np

INF = math.inf


def _flag(oracle_mod, delay_dist, dt_ms=0.1, idx=0):
    r = oracle_mod.eval_synapse((0, 10), (0, 10), oracle_mod.FIXED_TOTAL_NUMBER, 1, 0.0, (1.0, 0.0, -INF, INF),
                                delay_dist, 5, 0, dt_ms, idx)
    return r["boundary"], r["delay"], r["x"]


def test_exact_half_is_flagged(oracle_mod):
    """0.25 ms at dt = 0.1 ms: inv_dt = 1/0.1 = 10.0 exactly in fp64, x = 2.5 exactly -> k + 1/2 -> flag 1,
    and round half up gives 3 steps (Q5)."""
    assert 1.0 / 0.1 == 10.0
    b, d, x = _flag(oracle_mod, (0.25, 0.0, -INF, INF))
    assert x == 2.5 and b == 1 and d == 3
    # another exact half with a different resolution: 0.375 ms at dt = 0.25 ms -> x = 1.5
    b, d, x = _flag(oracle_mod, (0.375, 0.0, -INF, INF), dt_ms=0.25)
    assert x == 1.5 and b == 1 and d == 2


def test_band_is_1e_minus_9_wide_on_both_sides(oracle_mod):
    """x = 2.5 +- delta: flagged for delta = 5e-10, not for 2e-9, 1e-6, 1e-3 (a band of 1e-3 or 1e-6 fails here)."""
    for sign in (+1.0, -1.0):
        for delta, want in ((5e-10, 1), (2e-9, 0), (1e-6, 0), (1e-3, 0), (0.25, 0)):
            d_ms = (2.5 + sign * delta) / 10.0
            b, _, x = _flag(oracle_mod, (d_ms, 0.0, -INF, INF))
            assert abs(abs(x - 2.5) - delta) < 1e-12, (sign, delta, x)  # the constant lands where intended
            assert b == want, (sign, delta, x, b)


def test_integers_and_far_values_are_not_flagged(oracle_mod):
    for d_ms in (0.1, 0.2, 1.5, 0.26, 0.24, 3.14159, 6000.0):
        b, _, _ = _flag(oracle_mod, (d_ms, 0.0, -INF, INF))
        assert b == 0, d_ms


def test_exact_clamp_is_not_flagged(oracle_mod):
    """A value clipped TO the bound equals the bound: d_ms == lo -> not a boundary (the GPU clamps to the same
    constant); likewise hi."""
    b, d, x = _flag(oracle_mod, (0.03, 0.0, 0.1, INF))     # mean below lo -> d_ms = lo = 0.1 -> x = 1.0
    assert x == 1.0 and b == 0 and d == 1
    b, d, x = _flag(oracle_mod, (9.0, 0.0, -INF, 2.0))     # mean above hi -> d_ms = hi
    assert x == 20.0 and b == 0 and d == 20
    b, _, _ = _flag(oracle_mod, (0.1, 0.0, 0.1, INF))      # mean == lo exactly
    assert b == 0


def test_near_clip_bound_but_not_equal_is_flagged(oracle_mod):
    """d_ms within 1e-12 relative of lo (or hi) without being equal: the fp32/fp64 paths may fall on either side
    of the clamp -> flag 1.  1e-11 away -> flag 0 (x = 1.0 or 20.0 is far from a half)."""
    lo = 0.1
    near, far = lo * (1.0 + 5e-13), lo * (1.0 + 1e-11)
    assert near != lo and abs(near - lo) <= 1e-12 * lo < abs(far - lo)
    assert _flag(oracle_mod, (near, 0.0, lo, INF))[0] == 1
    assert _flag(oracle_mod, (far, 0.0, lo, INF))[0] == 0
    hi = 2.0
    near, far = hi * (1.0 - 4e-13), hi * (1.0 - 1e-11)
    assert near != hi and abs(near - hi) <= 1e-12 * hi < abs(far - hi)
    assert _flag(oracle_mod, (near, 0.0, -INF, hi))[0] == 1
    assert _flag(oracle_mod, (far, 0.0, -INF, hi))[0] == 0
    # infinite bounds never flag
    assert _flag(oracle_mod, (1.23, 0.0, -INF, INF))[0] == 0


def test_random_draws_are_almost_never_flagged(oracle_mod):
    """400,000 draws of the configs' delay distribution N(1.5, 0.75) clipped at 0.1 ms: the band around the halves
    has total relative width 2e-9, the clip band 1e-13 -> expected number of flags 8e-4.  Zero must be seen; a band of
    1e-6 would already give ~0.8 expected and 1e-3 hundreds."""
    o = oracle_mod.Oracle(dt_ms=0.1)
    o.create_population(1000)
    n = 400_000
    o.connect((0, 1000), (0, 1000), oracle_mod.FIXED_TOTAL_NUMBER, degree_or_total=n, weight=(1.0, 0.0, -INF, INF),
              delay_ms=(1.5, 0.75, 0.1, INF), seed=77)
    c = o.connections()
    assert c["boundary"].shape == (n,) and int(c["boundary"].sum()) == 0
    # about 3 % of the draws are clipped to exactly 0.1 ms (Phi(-1.87)): exact clamps, one step, not flagged
    clipped = int((c["delay"] == 1).sum())
    assert 0.02 * n < clipped < 0.06 * n
    o.close()


def test_flag_follows_the_connection_into_the_sorted_view(oracle_mod):
    """Two projections, one on an exact half (all flagged) and one not: the sorted view's flags are the
    creation-order flags gathered by perm."""
    o = oracle_mod.Oracle(dt_ms=0.1)
    o.create_population(50)
    o.connect((0, 50), (0, 50), oracle_mod.FIXED_TOTAL_NUMBER, degree_or_total=300, delay_ms=(0.25, 0.0, -INF, INF), seed=1)
    o.connect((0, 50), (0, 50), oracle_mod.FIXED_TOTAL_NUMBER, degree_or_total=500, delay_ms=(0.3, 0.0, -INF, INF), seed=1)
    u = o.connections(sorted=False)
    assert np.all(u["boundary"][:300] == 1) and np.all(u["boundary"][300:] == 0)
    o.finalize()
    s = o.connections(sorted=True)
    assert np.array_equal(s["boundary"], u["boundary"][s["perm"]])
    assert int(s["boundary"].sum()) == 300
    o.close()
