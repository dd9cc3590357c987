"""Pins of the spike-delivery oracle (oracle/delivery.cpp).  The queue / group machinery must reproduce
the plain definition of delayed delivery, evaluated here from the creation-order connections with no queue and no
index: a spike of multiplicity m emitted by node s in step k adds m * w_c to the input of target_c in step
k + delay_c, for every connection c with source s.  Plus hand-computed small cases."""
import numpy as np
import pytest

from paper_2306_09855_b200 import workloads as WL

INF = float("inf")


def _build(oracle_mod, net):
    o = oracle_mod.Oracle(dt_ms=net.dt_ms)
    WL.run(net, o)
    return o


def _raster(rng, n_nodes, steps, rate, max_mult=3):
    out = []
    for _ in range(steps):
        k = rng.binomial(n_nodes, rate)
        nodes = rng.choice(n_nodes, size=k, replace=False).astype(np.uint32)
        out.append((nodes, rng.integers(1, max_mult + 1, size=k).astype(np.uint32)))
    return out


def _definition(conn, n_nodes, raster, total_steps):
    """input_by_step[k][t] straight from the definition (creation-order arrays, fp64)."""
    by_src = {}
    order = np.argsort(conn["source"], kind="stable")
    src = conn["source"][order]
    bounds = np.searchsorted(src, np.arange(n_nodes + 1))
    res = np.zeros((total_steps, n_nodes))
    for k, (nodes, mult) in enumerate(raster):
        for s, m in zip(nodes, mult):
            c = order[bounds[s]:bounds[s + 1]]
            for tgt, w, d in zip(conn["target"][c], conn["weight"][c], conn["delay"][c]):
                if k + d < total_steps:
                    res[k + d, tgt] += float(w) * float(m)
    return res


def test_delivery_matches_the_definition_of_delayed_delivery(oracle_mod):
    net = WL.config0_tiny()  # 100 nodes, 1,000 connections, delays 1 .. ~40 steps
    o = _build(oracle_mod, net)
    conn = o.connections(sorted=False)
    rng = np.random.default_rng(7)
    steps, tail = 60, 70
    raster = _raster(rng, net.n_nodes, steps, 0.05)
    want = _definition(conn, net.n_nodes, raster, steps + tail)
    d = oracle_mod.Delivery(o)
    events = 0
    for k in range(steps + tail):
        nodes, mult = raster[k] if k < steps else (np.zeros(0, np.uint32), np.zeros(0, np.uint32))
        got = np.zeros(net.n_nodes)
        d.step(nodes, mult, got)
        np.testing.assert_allclose(got, want[k], rtol=1e-12, atol=1e-9, err_msg=f"step {k}")
        g, m = d.spike_array()
        events += sum(1 for _ in g)
    buffered, delivered = d.counts()
    assert buffered == 0, "every spike must have left its queue after the longest delay"
    # every emitted spike visits every group of its source exactly once
    idx = o.index()
    assert events == sum(int(idx["group_count"][s]) for nodes, _ in raster for s in nodes)
    assert delivered == sum(int(idx["src_offsets"][s + 1] - idx["src_offsets"][s]) for nodes, _ in raster for s in nodes)
    d.close()
    o.close()


def test_hand_computed_two_connections(oracle_mod):
    """node 0 -> node 1 with constant weight 2.5 and delay 3 steps (one_to_one on a 1-node range), emitted in step 0
    with multiplicity 2 and in step 1 with multiplicity 1: input[1] = 5.0 in step 3, 2.5 in step 4, nothing else."""
    o = oracle_mod.Oracle(dt_ms=0.1)
    a = o.create_population(1)
    b = o.create_population(1)
    o.connect((a, 1), (b, 1), oracle_mod.ONE_TO_ONE, weight=(2.5, 0.0, -INF, INF), delay_ms=(0.3, 0.0, -INF, INF), seed=1)
    o.finalize()
    d = oracle_mod.Delivery(o)
    seen = []
    for k in range(7):
        inp = np.zeros(2)
        if k == 0:
            d.step([0], [2], inp)
        elif k == 1:
            d.step([0, 1], None, inp)  # node 1 has no outgoing connection: buffers nothing
        else:
            d.step([], None, inp)
        seen.append(inp.copy())
        g, m = d.spike_array()
        assert list(g) == ([0] if k in (3, 4) else []) and list(m) == ({3: [2], 4: [1]}.get(k, []))
    want = np.zeros((7, 2))
    want[3, 1], want[4, 1] = 5.0, 2.5
    assert np.array_equal(np.array(seen), want)
    assert d.counts() == (0, 2)
    with pytest.raises(oracle_mod.OracleError):
        d.step([2], None, np.zeros(2))
    d.close()
    o.close()


def test_groups_mature_in_ascending_delay_order(oracle_mod):
    """One source with many connections: the spike array of the steps after one spike lists the source's groups one
    per matured delay, in the order of group_delay."""
    net = WL.Network("one_source", [1, 50], [WL.Projection(0, 1, "fixed_outdegree", 400, 0.0, (1.0, 0.0, -INF, INF),
                                                           (1.5, 0.75, 0.1, INF), 3)], 0.1)
    o = _build(oracle_mod, net)
    idx = o.index()
    d = oracle_mod.Delivery(o)
    order = []
    for k in range(80):
        inp = np.zeros(net.n_nodes)
        d.step([0] if k == 0 else [], None, inp)
        g, _ = d.spike_array()
        assert g.size <= 1
        if g.size:
            order.append((k, int(g[0])))
    G = int(idx["group_count"][0])
    assert [g for _, g in order] == list(range(G))
    assert [k for k, _ in order] == [int(x) for x in idx["group_delay"][:G]]
    d.close()
    o.close()


def test_delivery_with_receptor_ports_matches_the_definition(oracle_mod):
    """Connections created under nc/oc_set_connection_attributes(port) deliver into the input of (port, target)
    (reading F2): the plain definition evaluated per port from the creation-order arrays."""
    o = oracle_mod.Oracle(dt_ms=0.1)
    o.create_population(40)
    W, D = (5.0, 1.0, 0.0, INF), (1.0, 0.5, 0.1, INF)
    ports = [0, 2, 1, 2]
    for k, port in enumerate(ports):
        o.set_connection_attributes(port)
        o.connect((0, 40), (0, 40), oracle_mod.FIXED_TOTAL_NUMBER, degree_or_total=300, weight=W, delay_ms=D, seed=3 + k)
    conn = o.connections(sorted=False)
    port_of = o.read_connection_attributes(sorted=False)[0]
    assert np.array_equal(port_of, np.repeat(np.array(ports, np.uint8), 300))
    o.finalize()
    rng = np.random.default_rng(11)
    steps, tail = 30, 40
    raster = _raster(rng, 40, steps, 0.1)
    want = np.zeros((steps + tail, 3, 40))
    for p in range(3):
        sel = port_of == p
        sub = {f: conn[f][sel] for f in ("source", "target", "weight", "delay")}
        want[:, p, :] = _definition(sub, 40, raster, steps + tail)
    d = oracle_mod.Delivery(o)
    assert d.n_ports == 3
    for k in range(steps + tail):
        nodes, mult = raster[k] if k < steps else (np.zeros(0, np.uint32), np.zeros(0, np.uint32))
        got = np.zeros(3 * 40)
        d.step(nodes, mult, got)
        np.testing.assert_allclose(got.reshape(3, 40), want[k], rtol=1e-12, atol=1e-9, err_msg=f"step {k}")
    d.close(); o.close()
