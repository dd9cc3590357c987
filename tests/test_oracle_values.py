"""Pins of per-connection value arrays in the oracle (weights and delays can "be specified for each
connection by an array having a size equal to the number of connections"; delays are divided by the time step, rounded,
at least one step)."""
import numpy as np
import pytest

INF = float("inf")
W = (20.0, 2.0, 0.0, INF)
D = (1.5, 0.75, 0.1, INF)


def _build(oracle_mod, rule, kw, weights=None, delays=None, dt=0.1, src=(0, 40), tgt=(40, 60)):
    o = oracle_mod.Oracle(dt_ms=dt)
    o.create_population(100)
    o.connect(src, tgt, rule, weight=W, delay_ms=D, seed=11, weights=weights, delays=delays, **kw)
    c = o.connections(sorted=False)
    o.close()
    return c


def test_values_pass_through_and_everything_else_is_unchanged(oracle_mod):
    """Entry i belongs to connection i (Eq. 2); sources, targets and the parameter that has no array are exactly
    those of the distribution form with the same seed and projection id."""
    rng = np.random.default_rng(0)
    for rule, kw, n in ((oracle_mod.FIXED_TOTAL_NUMBER, dict(degree_or_total=777), 777),
                        (oracle_mod.FIXED_INDEGREE, dict(degree_or_total=5), 300),
                        (oracle_mod.FIXED_OUTDEGREE, dict(degree_or_total=3), 120),
                        (oracle_mod.ALL_TO_ALL, {}, 2400)):
        base = _build(oracle_mod, rule, kw)
        assert base["n"] == n
        w = rng.normal(size=n).astype(np.float32)
        d = rng.uniform(0.1, 5.0, size=n)
        both = _build(oracle_mod, rule, kw, weights=w, delays=d)
        only_w = _build(oracle_mod, rule, kw, weights=w)
        only_d = _build(oracle_mod, rule, kw, delays=d)
        for c in (both, only_w, only_d):
            assert np.array_equal(c["source"], base["source"]) and np.array_equal(c["target"], base["target"])
        assert np.array_equal(both["weight"], w) and np.array_equal(only_w["weight"], w)
        assert np.array_equal(only_w["delay"], base["delay"]) and np.array_equal(only_d["weight"], base["weight"])
        assert np.array_equal(both["delay"], only_d["delay"])


def test_delay_conversion_hand_cases(oracle_mod):
    """dt = 0.1 ms: 0.04 -> 0.4 -> 0 -> at least 1; 0.15 -> 1.5 -> 2 (half up); 0.25 -> 3; 1.0 -> 10; 0 and negative
    -> 1; 0.1499 -> 1; 6553.5 -> 65535.  dt = 0.25 ms: 1.0 -> 4, 0.3 -> 1.2 -> 1, 0.4 -> 1.6 -> 2."""
    d = np.array([0.04, 0.15, 0.25, 1.0, 0.0, -3.0, 0.1499, 6553.5])
    c = _build(oracle_mod, oracle_mod.ONE_TO_ONE, {}, delays=d, src=(0, 8), tgt=(8, 8))
    assert c["delay"].tolist() == [1, 2, 3, 10, 1, 1, 1, 65535]
    c = _build(oracle_mod, oracle_mod.ONE_TO_ONE, {}, delays=np.array([1.0, 0.3, 0.4]), dt=0.25, src=(0, 3), tgt=(8, 3))
    assert c["delay"].tolist() == [4, 1, 2]


def test_delay_conversion_against_numpy_and_order(oracle_mod):
    """floor(d / dt + 1/2) evaluated with numpy on values away from rounding boundaries, and the organised order of
    the result: sorted by (source, given delay), ties in creation order."""
    rng = np.random.default_rng(3)
    n = 5000
    d = (rng.integers(1, 400, size=n) + rng.uniform(-0.4, 0.4, size=n)) * 0.1  # never within 0.1 step of a boundary
    o = oracle_mod.Oracle(dt_ms=0.1)
    o.create_population(50)
    o.connect((0, 50), (0, 50), oracle_mod.FIXED_TOTAL_NUMBER, degree_or_total=n, weight=W, delay_ms=D, seed=2, delays=d)
    o.finalize()
    u, s = o.connections(sorted=False), o.connections(sorted=True)
    want = np.maximum(1, np.floor(d / 0.1 + 0.5)).astype(np.uint16)
    assert np.array_equal(u["delay"], want)
    perm = np.argsort((u["source"].astype(np.uint64) << np.uint64(16)) | want.astype(np.uint64), kind="stable")
    assert np.array_equal(s["perm"], perm.astype(np.uint32)) and np.array_equal(s["delay"], want[perm])
    o.close()


def test_bad_value_arrays_are_rejected_and_leave_the_context_unchanged(oracle_mod):
    o = oracle_mod.Oracle(dt_ms=0.1)
    o.create_population(20)
    E = oracle_mod.ERR_INVALID_ARG
    ftn = dict(degree_or_total=10)
    assert o.connect_rc((0, 20), (0, 20), oracle_mod.FIXED_TOTAL_NUMBER, weights=np.zeros(9), **ftn) == E      # size
    assert o.connect_rc((0, 20), (0, 20), oracle_mod.FIXED_TOTAL_NUMBER, delays=np.zeros(11), **ftn) == E
    assert o.connect_rc((0, 20), (0, 20), oracle_mod.FIXED_TOTAL_NUMBER, delays=np.full(10, np.nan), **ftn) == E
    assert o.connect_rc((0, 20), (0, 20), oracle_mod.FIXED_TOTAL_NUMBER, delays=np.full(10, np.inf), **ftn) == E
    assert o.connect_rc((0, 20), (0, 20), oracle_mod.FIXED_TOTAL_NUMBER, weights=np.full(10, np.nan), **ftn) == E
    assert o.connect_rc((0, 20), (0, 20), oracle_mod.PAIRWISE_BERNOULLI, p=0.5, weights=np.zeros(200)) == E  # no count
    assert o.connect_rc((0, 20), (0, 20), oracle_mod.FIXED_TOTAL_NUMBER, delays=np.full(10, 6553.6), **ftn) == oracle_mod.ERR_CAPACITY
    assert o.num_connections() == 0 and o.num_blocks() == 0
    # the projection id was not consumed: the next call draws what a first call draws
    o.connect((0, 20), (0, 20), oracle_mod.FIXED_TOTAL_NUMBER, weight=W, delay_ms=D, seed=5, **ftn)
    p = oracle_mod.Oracle(dt_ms=0.1)
    p.create_population(20)
    p.connect((0, 20), (0, 20), oracle_mod.FIXED_TOTAL_NUMBER, weight=W, delay_ms=D, seed=5, **ftn)
    a, b = o.connections(sorted=False), p.connections(sorted=False)
    assert np.array_equal(a["source"], b["source"]) and np.array_equal(a["weight"], b["weight"])
    o.close(); p.close()
