"""Pins of the oracle's shard filter (reading S1: a context keeps the connections whose target it owns): against the
UNSHARDED oracle -- the shards partition its connections, each in the unsharded order, creation order and organised order
alike (a stable sort commutes with taking a subsequence); per-source out-degrees add up; Eq. 1 over what is held."""
import math

import numpy as np
import pytest

import oracle as O

W, D = (20.0, 2.0, 0.0, math.inf), (1.5, 0.75, 0.1, math.inf)
R = dict(one_to_one=0, all_to_all=1, fixed_indegree=2, fixed_outdegree=3, fixed_total_number=4, pairwise_bernoulli=5)
N = 240


def recipe(o):
    rng = np.random.default_rng(4)
    arr = rng.permutation(N)[:90].astype(np.uint32)
    o.connect((0, 120), (60, 120), R["fixed_total_number"], degree_or_total=9000, weight=W, delay_ms=D, seed=1)
    o.connect((0, 100), (100, 100), R["one_to_one"], weight=W, delay_ms=D, seed=2)
    o.connect((10, 40), (0, 240), R["all_to_all"], weight=W, delay_ms=D, seed=3)
    o.set_rule_flags(O.NO_AUTAPSES | O.NO_MULTAPSES)
    o.connect((0, 240), (0, 240), R["fixed_indegree"], degree_or_total=20, weight=W, delay_ms=D, seed=4)
    o.set_rule_flags(O.NO_AUTAPSES)
    o.connect(arr, (0, 200), R["pairwise_bernoulli"], p=0.2, weight=W, delay_ms=D, seed=5)
    o.set_rule_flags(0)
    o.connect((0, 50), arr, R["fixed_outdegree"], degree_or_total=30, weight=W, delay_ms=D, seed=6,
              weights=rng.normal(0, 3, 50 * 30).astype(np.float32))


def build(shard=None, B=1000):
    o = O.Oracle(dt_ms=0.1, block_size=B)
    o.create_population(N)
    if shard is not None:
        o.set_shard(*shard)
    recipe(o)
    cu = {k: np.array(v) for k, v in o.connections(sorted=False).items() if k in ("source", "target", "weight", "delay")}
    nb = o.num_blocks()
    o.finalize()
    cs = {k: np.array(v) for k, v in o.connections(sorted=True).items() if k in ("source", "target", "weight", "delay", "perm")}
    idx = o.index()
    outd = np.array(o.degree_histogram(1)[0])
    o.close()
    return cu, cs, idx, outd, nb


@pytest.mark.parametrize("world", [1, 2, 3, 7])
def test_shards_partition_the_unsharded_network_in_its_own_order(world):
    fu, fs, fidx, foutd, _ = build()
    bounds = [N * r // world for r in range(world + 1)]
    total, outd_sum = 0, np.zeros(N, dtype=np.int64)
    for r in range(world):
        first, count = bounds[r], bounds[r + 1] - bounds[r]
        cu, cs, idx, outd, nb = build((first, count))
        own_u = (fu["target"] >= first) & (fu["target"] < first + count)
        own_s = (fs["target"] >= first) & (fs["target"] < first + count)
        for k in ("source", "target", "weight", "delay"):
            assert np.array_equal(cu[k], fu[k][own_u]), (world, r, k, "creation order")
            assert np.array_equal(cs[k], fs[k][own_s]), (world, r, k, "organised order")
        # the shard's permutation refers to ITS creation positions: rank of the global position among the owned ones
        rank_of = np.cumsum(own_u) - 1
        assert np.array_equal(cs["perm"], rank_of[fs["perm"][own_s]])
        assert nb == (cu["source"].size + 999) // 1000
        assert idx["src_offsets"][-1] == cu["source"].size
        total += cu["source"].size
        outd_sum += outd
    assert total == fu["source"].size and np.array_equal(outd_sum, foutd)
    if world == 1:
        assert np.array_equal(idx["group_start"], fidx["group_start"])


def test_set_shard_only_before_the_first_connect():
    o = O.Oracle(dt_ms=0.1)
    o.create_population(10)
    o.connect((0, 10), (0, 10), R["all_to_all"], weight=W, delay_ms=D)
    with pytest.raises(O.OracleError):
        o.set_shard(0, 5)
    o.close()
