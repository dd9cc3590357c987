"""Pins of the receptor port / synaptic group fields of a connection in the oracle: they belong to the
connect calls issued while they are in force, travel with their connection into the organised order, and change
nothing else."""
import numpy as np

INF = float("inf")
W = (20.0, 2.0, 0.0, INF)
D = (1.5, 0.75, 0.1, INF)


def _net(oracle_mod, with_attrs):
    o = oracle_mod.Oracle(dt_ms=0.1, block_size=64)
    o.create_population(30)
    sizes = []
    for k, (port, group) in enumerate([(0, 0), (3, 0), (255, 7), (1, 1)]):
        if with_attrs:
            o.set_connection_attributes(port, group)
        rule = [oracle_mod.FIXED_TOTAL_NUMBER, oracle_mod.ALL_TO_ALL, oracle_mod.PAIRWISE_BERNOULLI, oracle_mod.FIXED_INDEGREE][k]
        before = o.num_connections()
        o.connect((0, 30), (0, 30), rule, degree_or_total=[500, 0, 0, 4][k], p=0.3, weight=W, delay_ms=D, seed=77)
        sizes.append(o.num_connections() - before)
    return o, sizes


def test_attributes_follow_their_projection_and_their_connection(oracle_mod):
    o, sizes = _net(oracle_mod, True)
    want_p = np.repeat(np.array([0, 3, 255, 1], np.uint8), sizes)
    want_g = np.repeat(np.array([0, 0, 7, 1], np.uint8), sizes)
    port, group = o.read_connection_attributes(sorted=False)
    assert np.array_equal(port, want_p) and np.array_equal(group, want_g)
    o.finalize()
    perm = o.connections(sorted=True)["perm"]
    port_s, group_s = o.read_connection_attributes(sorted=True)
    assert np.array_equal(port_s, want_p[perm]) and np.array_equal(group_s, want_g[perm])
    # a slice of the organised view
    p2, g2 = o.read_connection_attributes(sorted=True, first=100, count=250)
    assert np.array_equal(p2, port_s[100:350]) and np.array_equal(g2, group_s[100:350])
    o.close()


def test_attributes_change_nothing_else(oracle_mod):
    a, _ = _net(oracle_mod, True)
    b, _ = _net(oracle_mod, False)
    for o in (a, b):
        o.finalize()
    ca, cb = a.connections(sorted=True), b.connections(sorted=True)
    for f in ("source", "target", "weight", "delay", "perm"):
        assert np.array_equal(ca[f], cb[f]), f
    pb, gb = b.read_connection_attributes(sorted=True)
    assert not pb.any() and not gb.any()  # the default is port 0, group 0 (static synapses)
    a.close(); b.close()
