"""Pins for the oracle's organisation step (readings D10-D12; Eq. 14): the sort
against numpy's stable sort (library routine = the plain definition), the index against a brute-force
dict/set construction on small networks, plus the invariants of SURVEY.md 8(c).  CPU only."""
import math

import numpy as np
import pytest

from paper_2306_09855_b200 import workloads as WL

INF = math.inf


def _build(oracle_mod, net, B=0):
    o = oracle_mod.Oracle(dt_ms=net.dt_ms, block_size=B)
    WL.run(net, o)
    return o


def _brute_index(src, delay, n_nodes):
    """Plain-Python construction straight from PAPER.md:121-132."""
    n = len(src)
    out_degree = [0] * n_nodes
    for s in src:
        out_degree[s] += 1
    groups = {}  # source -> sorted set of delays
    for s, d in zip(src, delay):
        groups.setdefault(int(s), set()).add(int(d))
    G = [len(groups.get(s, ())) for s in range(n_nodes)]
    p = [0] * (n_nodes + 1)
    for s in range(n_nodes):
        p[s + 1] = p[s] + G[s]  # Eq. 14
    off = [0] * (n_nodes + 1)
    for s in range(n_nodes):
        off[s + 1] = off[s] + out_degree[s]
    start, gdelay = [], []
    for s in range(n_nodes):
        pos = off[s]
        for d in sorted(groups.get(s, ())):
            start.append(pos)
            gdelay.append(d)
            pos += sum(1 for ss, dd in zip(src, delay) if ss == s and dd == d) if n < 4000 else 0
    return out_degree, off, G, p, start, gdelay


@pytest.mark.parametrize("B", [0, 10, 64])
def test_config0_sort_and_index(oracle_mod, B):
    net = WL.config0_tiny()
    o = _build(oracle_mod, net, B=B)
    assert o.num_connections() == 1000 and o.num_nodes() == 100
    assert o.num_blocks() == (-(-1000 // B) if B else 1)
    c, s = o.connections(), o.connections(sorted=True)
    key = (c["source"].astype(np.uint64) << np.uint64(16)) | c["delay"].astype(np.uint64)
    perm = np.argsort(key, kind="stable")
    assert np.array_equal(s["perm"], perm.astype(np.uint32))
    assert np.array_equal(np.lexsort((np.arange(1000), c["delay"], c["source"])), perm)
    for k in ("source", "target", "weight", "delay"):
        assert np.array_equal(s[k], c[k][perm])
    idx = o.index()
    od, off, G, p, start, gdelay = _brute_index(s["source"].tolist(), s["delay"].tolist(), 100)
    assert idx["src_offsets"].tolist() == off
    assert idx["group_count"].tolist() == G
    assert idx["group_ptr"].tolist() == p
    assert idx["total_groups"] == p[-1] == len(start)
    assert idx["group_start"].tolist() == start
    assert idx["group_delay"].tolist() == gdelay
    outdeg, mx = o.degree_histogram(1)
    assert outdeg.tolist() == od and mx == max(od)
    indeg, _ = o.degree_histogram(0)
    assert indeg.tolist() == np.bincount(c["target"], minlength=100).tolist()
    # config 0: every E neuron has in-degree 8 + 2 and every I neuron too (fixed_indegree)
    assert set(indeg.tolist()) == {10}


def test_sort_invariants_medium(oracle_mod):
    """SURVEY.md 8(c) sort/index pins on a network with empty sources, multapses and three rules."""
    o = oracle_mod.Oracle(dt_ms=0.1)
    a = o.create_population(300)
    b = o.create_population(200)
    c_ = o.create_population(50)  # never a source
    W, D = (20.0, 2.0, 0.0, INF), (1.5, 0.75, 0.1, INF)
    o.connect((a, 300), (b, 200), oracle_mod.FIXED_TOTAL_NUMBER, degree_or_total=20000, weight=W, delay_ms=D, seed=5)
    o.connect((b, 200), (c_, 50), oracle_mod.FIXED_OUTDEGREE, degree_or_total=30, weight=W, delay_ms=D, seed=5)
    o.connect((a + 10, 100), (a, 300), oracle_mod.PAIRWISE_BERNOULLI, p=0.2, weight=W, delay_ms=D, seed=5)
    o.finalize()
    c, s, idx = o.connections(), o.connections(sorted=True), o.index()
    n, N = c["n"], 550
    assert sorted(s["perm"].tolist()) == list(range(n))  # a permutation
    key = (s["source"].astype(np.int64) << 16) | s["delay"]
    assert np.all(np.diff(key) >= 0)  # sorted by (source, delay)
    same = np.diff(key) == 0
    assert np.all(np.diff(s["perm"].astype(np.int64))[same] > 0)  # stable: ties keep creation order
    okey = (c["source"].astype(np.uint64) << np.uint64(16)) | c["delay"].astype(np.uint64)
    assert np.array_equal(s["perm"], np.argsort(okey, kind="stable").astype(np.uint32))
    off, gp, gs, gd, G = idx["src_offsets"], idx["group_ptr"], idx["group_start"], idx["group_delay"], idx["group_count"]
    assert off[0] == 0 and off[N] == n and len(off) == N + 1
    assert np.array_equal(np.diff(off.astype(np.int64)), np.bincount(c["source"], minlength=N))
    assert G.sum() == idx["total_groups"] == gp[N] and gp[0] == 0
    assert np.array_equal(np.diff(gp.astype(np.int64)), G)
    assert np.all(np.diff(gs.astype(np.int64)) > 0)  # strictly increasing
    heads = np.concatenate(([True], np.diff(key) != 0))
    assert np.array_equal(np.flatnonzero(heads), gs)  # every entry a head, every head present
    assert np.array_equal(gd, s["delay"][gs])
    for node in range(N):
        if G[node] > 0:
            assert gs[gp[node]] == off[node]
        else:
            assert off[node + 1] == off[node]
    assert np.all(G[500:] == 0)
    # groups per source = number of distinct delays of that source (set definition)
    for node in (0, 17, 299, 300, 420):
        sel = c["source"] == node
        assert G[node] == len(set(c["delay"][sel].tolist()))


def test_empty_network_finalize(oracle_mod):
    o = oracle_mod.Oracle(dt_ms=0.1)
    o.create_population(5)
    o.finalize()
    idx = o.index()
    assert idx["total_groups"] == 0 and idx["src_offsets"].tolist() == [0] * 6 and idx["group_ptr"].tolist() == [0] * 6
    assert o.connections(sorted=True)["n"] == 0


def test_sorted_view_requires_finalize(oracle_mod):
    o = oracle_mod.Oracle(dt_ms=0.1)
    o.create_population(5)
    with pytest.raises(oracle_mod.OracleError):
        o.connections(sorted=True)
    with pytest.raises(oracle_mod.OracleError):
        o.index()
