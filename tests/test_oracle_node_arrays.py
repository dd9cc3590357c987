"""Pins of the explicit-node-array form of connect in the oracle ("the above formulas are used to derive
the indexes of the array elements from which to extract the node indexes")."""
import numpy as np
import pytest

INF = float("inf")
W = (20.0, 2.0, 0.0, INF)
D = (1.5, 0.75, 0.1, INF)


def _conn(o):
    return o.connections(sorted=False)


def test_identity_arrays_reproduce_the_range_form(oracle_mod):
    """arrays that list a consecutive range give exactly what the range form gives (same projection id, same seed)"""
    for rule, kw in ((oracle_mod.FIXED_TOTAL_NUMBER, dict(degree_or_total=5000)), (oracle_mod.FIXED_INDEGREE, dict(degree_or_total=7)),
                     (oracle_mod.FIXED_OUTDEGREE, dict(degree_or_total=9)), (oracle_mod.ALL_TO_ALL, {}),
                     (oracle_mod.PAIRWISE_BERNOULLI, dict(p=0.3))):
        a, b = oracle_mod.Oracle(), oracle_mod.Oracle()
        for o in (a, b):
            o.create_population(50)
            o.create_population(70)
        a.connect((10, 30), (50, 60), rule, weight=W, delay_ms=D, seed=9, **kw)
        b.connect(np.arange(10, 40), np.arange(50, 110), rule, weight=W, delay_ms=D, seed=9, **kw)
        ca, cb = _conn(a), _conn(b)
        assert ca["n"] == cb["n"] and ca["n"] > 0
        for k in ("source", "target", "weight", "delay"):
            assert np.array_equal(ca[k], cb[k]), (rule, k)


def test_one_to_one_and_all_to_all_closed_forms_through_arrays(oracle_mod):
    """Eqs. 4-7 with array lookup: one_to_one pairs element i of both arrays; all_to_all pairs element i div N_tgt of
    the source array with element i mod N_tgt of the target array.  Ids may repeat and need not be sorted."""
    o = oracle_mod.Oracle()
    o.create_population(100)
    src = np.array([90, 3, 3, 41, 7], dtype=np.uint32)
    tgt = np.array([5, 99, 0, 5, 62], dtype=np.uint32)
    o.connect(src, tgt, oracle_mod.ONE_TO_ONE, weight=W, delay_ms=D, seed=1)
    c = _conn(o)
    assert list(c["source"]) == list(src) and list(c["target"]) == list(tgt)
    o.connect(src, tgt[:3], oracle_mod.ALL_TO_ALL, weight=W, delay_ms=D, seed=1)
    c = _conn(o)
    i = np.arange(15)
    assert list(c["source"][5:]) == list(src[i // 3]) and list(c["target"][5:]) == list(tgt[:3][i % 3])
    o.close()


def test_mixed_range_and_array_and_random_rule_statistics(oracle_mod):
    """fixed_indegree from an array of 4 source ids onto a target range: every target gets exactly K connections
    (Eq. 11) and only listed ids appear, each about a quarter of the time."""
    o = oracle_mod.Oracle()
    o.create_population(1000)
    ids = np.array([17, 500, 501, 999], dtype=np.uint32)
    o.connect(ids, (100, 200), oracle_mod.FIXED_INDEGREE, degree_or_total=50, weight=W, delay_ms=D, seed=3)
    c = _conn(o)
    assert c["n"] == 200 * 50
    assert np.array_equal(np.bincount(c["target"], minlength=1000)[100:300], np.full(200, 50))
    cnt = np.bincount(c["source"], minlength=1000)
    assert cnt.sum() == cnt[ids].sum()
    assert np.all(np.abs(cnt[ids] - 2500) < 5 * np.sqrt(10000 * 0.25 * 0.75))
    o.close()


def test_bad_ids_and_sizes_are_rejected(oracle_mod):
    o = oracle_mod.Oracle()
    o.create_population(10)
    assert o.connect_rc(np.array([1, 10]), (0, 10), oracle_mod.ALL_TO_ALL) == oracle_mod.ERR_INVALID_ARG
    assert o.connect_rc((0, 10), np.array([11]), oracle_mod.ALL_TO_ALL) == oracle_mod.ERR_INVALID_ARG
    assert o.connect_rc(np.array([1, 2, 3]), np.array([4, 5]), oracle_mod.ONE_TO_ONE) == oracle_mod.ERR_INVALID_ARG
    assert o.connect_rc(np.array([], dtype=np.uint32), (0, 10), oracle_mod.ALL_TO_ALL) == oracle_mod.ERR_INVALID_ARG
    assert o.num_connections() == 0
    # an array longer than the node count (ids repeat) is legal
    assert o.connect_rc(np.zeros(25, dtype=np.uint32), (0, 10), oracle_mod.ALL_TO_ALL) == oracle_mod.OK
    assert o.num_connections() == 250
    o.close()
