"""GPU parity of spike delivery (include/nc_delivery.h) against oracle/delivery.cpp on the same seeded spike
rasters: per step the spike array (as a multiset: its order on the device is arbitrary) must be identical, and the
input of every node must match the oracle's fp64 sum within the fp32 accumulation tolerance
|err| <= 1e-5 * max(1, max |input|) (sums of at most a few hundred terms of magnitude <= 400, fp32 atomics in arbitrary
order: relative error ~ sqrt(terms) * 6e-8)."""
import math

import numpy as np
import pytest

from paper_2306_09855_b200 import workloads as WL

pytestmark = pytest.mark.gpu
INF = math.inf


@pytest.fixture(scope="module")
def nc_mod():
    from paper_2306_09855_b200 import binding, build
    build.build()
    return binding


@pytest.fixture(params=["fused", "two_kernels"], autouse=True)
def delivery_form(request, monkeypatch):
    """every test runs over the cooperative one-launch step and over the two-kernel step (the fallback when cooperative
    launch is unavailable; nc_delivery_create reads NC_DELIVERY_TWO_KERNELS)"""
    monkeypatch.setenv("NC_DELIVERY_TWO_KERNELS", "1" if request.param == "two_kernels" else "0")
    return request.param


def _raster(rng, n_nodes, steps, rate, max_mult):
    out = []
    for _ in range(steps):
        k = int(rng.binomial(n_nodes, rate))
        nodes = rng.choice(n_nodes, size=k, replace=False).astype(np.uint32)
        out.append((nodes, rng.integers(1, max_mult + 1, size=k).astype(np.uint32)))
    return out


def _run_both(nc_mod, oracle_mod, net, steps, tail, rate, capacity, max_mult=3, use_mult=True, seed=11):
    import torch
    o = oracle_mod.Oracle(dt_ms=net.dt_ms)
    WL.run(net, o)
    g = nc_mod.NC(dt_ms=net.dt_ms)
    WL.run(net, g)
    od, gd = oracle_mod.Delivery(o), nc_mod.Delivery(g, capacity)
    rng = np.random.default_rng(seed)
    raster = _raster(rng, net.n_nodes, steps, rate, max_mult)
    inp = torch.zeros(net.n_nodes, dtype=torch.float32, device="cuda")
    worst = 0.0
    for k in range(steps + tail):
        nodes, mult = raster[k] if k < steps else (np.zeros(0, np.uint32), np.zeros(0, np.uint32))
        want = np.zeros(net.n_nodes)
        od.step(nodes, mult if use_mult else None, want)
        inp.zero_()
        tn = torch.from_numpy(nodes.astype(np.int32)).cuda()
        tm = torch.from_numpy(mult.astype(np.int32)).cuda() if use_mult else None
        gd.step(tn, tm, inp)
        got = inp.cpu().numpy().astype(np.float64)
        tol = 1e-5 * max(1.0, float(np.abs(want).max()))
        err = float(np.abs(got - want).max())
        assert err <= tol, f"step {k}: input error {err} > {tol}"
        worst = max(worst, err / tol)
        og, om = od.spike_array()
        gg, gm = gd.read_spike_array()
        assert np.array_equal(np.sort(og.astype(np.uint64) << np.uint64(32) | om), np.sort(gg.astype(np.uint64) << np.uint64(32) | gm)), f"step {k}: spike array"
    ob, oe = od.counts()
    c = gd.counts()
    assert c["buffered"] == ob and c["events"] == oe and c["dropped"] == 0 and c["bad_nodes"] == 0
    gd.close(); od.close(); g.close(); o.close()
    return worst, oe


def test_delivery_tiny_network_every_step(nc_mod, oracle_mod):
    worst, events = _run_both(nc_mod, oracle_mod, WL.config0_tiny(), steps=80, tail=70, rate=0.05, capacity=4096)
    assert events > 1000


def test_delivery_without_multiplicities(nc_mod, oracle_mod):
    _run_both(nc_mod, oracle_mod, WL.config0_tiny(), steps=40, tail=70, rate=0.1, capacity=4096, use_mult=False)


def test_delivery_microcircuit_scaled(nc_mod, oracle_mod):
    """configs[2] at 5 % of the populations (3,858 nodes, 7.5e5 connections, E and I delays): many groups per source,
    several warps' worth of connections per group, a few hundred spikes in flight."""
    worst, events = _run_both(nc_mod, oracle_mod, WL.config2_microcircuit(scale=0.05), steps=50, tail=65, rate=0.01,
                              capacity=1 << 16, seed=3)
    assert events > 3e5


def test_delivery_edge_cases(nc_mod, oracle_mod):
    import torch
    net = WL.config0_tiny()
    g = nc_mod.NC(dt_ms=net.dt_ms)
    firsts = WL.run(net, g, finalize=False)
    with pytest.raises(nc_mod.NCError) as e:  # before nc_finalize
        nc_mod.Delivery(g, 16)
    assert e.value.code == nc_mod.ERR_STATE
    g.finalize()
    with pytest.raises(nc_mod.NCError):
        nc_mod.Delivery(g, 0)
    d = nc_mod.Delivery(g, 4)  # room for four buffered spikes only
    inp = torch.zeros(net.n_nodes, dtype=torch.float32, device="cuda")
    d.step(torch.zeros(0, dtype=torch.int32, device="cuda"), None, inp)  # an empty step
    nodes = torch.tensor([0, 1, 2, 3, 4, 5, 1000], dtype=torch.int32, device="cuda")  # one id outside the network
    d.step(nodes, None, inp)
    c = d.counts()
    assert c["buffered"] == 4 and c["dropped"] == 2 and c["bad_nodes"] == 1
    mult0 = torch.zeros(3, dtype=torch.int32, device="cuda")
    d2 = nc_mod.Delivery(g, 64)
    d2.step(torch.tensor([7, 8, 9], dtype=torch.int32, device="cuda"), mult0, inp)  # multiplicity 0 = no spike
    assert d2.counts()["buffered"] == 0
    d.close(); d2.close(); g.close()


@pytest.mark.parametrize("copass", [False, True], ids=["flat", "blocks"])
def test_delivery_with_receptor_ports(nc_mod, oracle_mod, copass):
    """Projections with different receptor ports (nc_set_connection_attributes): every (port, node) input
    equals the oracle's, over the flat organised arrays and over COPASS-organised blocks."""
    import torch
    o = oracle_mod.Oracle(dt_ms=0.1, block_size=500)
    g = nc_mod.NC(dt_ms=0.1, block_size=500, flags=nc_mod.FLAG_ORGANISE_COPASS if copass else 0)
    W, D = (5.0, 1.0, 0.0, float("inf")), (1.0, 0.5, 0.1, float("inf"))
    for b in (o, g):
        b.create_population(60)
        for k, port in enumerate([0, 3, 1, 3, 0]):
            b.set_connection_attributes(port)
            b.connect((0, 60), (0, 60), 4, degree_or_total=700, weight=W, delay_ms=D, seed=20 + k)  # fixed_total_number
        b.finalize()
    od, gd = oracle_mod.Delivery(o), nc_mod.Delivery(g, 4096)
    assert gd.n_ports == od.n_ports == 4
    inp = torch.zeros(4 * 60, dtype=torch.float32, device="cuda")
    rng = np.random.default_rng(6)
    for k in range(70):
        nodes = rng.choice(60, size=int(rng.integers(0, 8)) if k < 30 else 0, replace=False).astype(np.uint32)
        want = np.zeros(4 * 60)
        od.step(nodes, None, want)
        inp.zero_()
        gd.step(torch.from_numpy(nodes.astype(np.int32)).cuda(), None, inp)
        got = inp.cpu().numpy()
        assert np.abs(got - want).max() <= 1e-5 * max(1.0, np.abs(want).max()), k
        assert not got.reshape(4, 60)[2].any()  # port 2 is unused
    assert gd.counts()["events"] == od.counts()[1] > 0
    gd.close(); od.close(); g.close(); o.close()


def test_run_equals_step_by_step(nc_mod):
    """nc_delivery_run over a raster known beforehand = the same steps issued one by one."""
    import torch
    net = WL.config0_tiny()
    rng = np.random.default_rng(9)
    counts = rng.integers(0, 9, size=50)
    offs = np.concatenate([[0], np.cumsum(counts)]).astype(np.uint64)
    nodes = np.concatenate([rng.choice(net.n_nodes, size=int(k), replace=False) for k in counts]).astype(np.int32)
    d_nodes = torch.from_numpy(nodes).cuda()
    res = []
    for mode in ("steps", "run"):
        g = nc_mod.NC(dt_ms=net.dt_ms)
        WL.run(net, g)
        d = nc_mod.Delivery(g, 4096)
        inp = torch.zeros(net.n_nodes, dtype=torch.float32, device="cuda")
        if mode == "steps":
            for k in range(50):
                d.step(d_nodes[int(offs[k]):int(offs[k + 1])], None, inp)
        else:
            d.run(d_nodes, None, offs, inp)
        res.append((inp.cpu().numpy(), d.counts(), sorted(zip(*[a.tolist() for a in d.read_spike_array()]))))
        d.close(); g.close()
    assert res[0][1] == res[1][1] and res[0][2] == res[1][2]
    assert np.abs(res[0][0] - res[1][0]).max() <= 1e-4 * max(1.0, np.abs(res[0][0]).max())  # fp32 atomics reorder


def test_context_cannot_be_destroyed_under_a_delivery(nc_mod):
    """nc_destroy refuses (NC_ERR_STATE, nothing freed) while a delivery object of the context exists; the binding's
    NC.close() closes its deliveries first."""
    import ctypes as C
    net = WL.config0_tiny()
    g = nc_mod.NC(dt_ms=net.dt_ms)
    WL.run(net, g)
    d = nc_mod.Delivery(g, 256)
    assert g._L.nc_destroy(g._h) == nc_mod.ERR_STATE  # raw call: the context stays alive and usable
    assert g.num_connections() == 1000
    g.close()            # closes d first, then the context
    assert not d._h
