"""Shared helpers of the GPU parity tests: build the same recipe on the CUDA path and on the oracle and
compare element by element.  The bar (BASELINE.json north_star): sources, targets, permutation and every
index array bit-exact; weights within 1e-5 relative (to the projection's weight scale); delays bit-exact
except that at most 1e-7 of the synapses may differ by one step, and only where the oracle flags a
rounding boundary (reading D8) -- every mismatch is counted and reported."""
import math

import numpy as np

from paper_2306_09855_b200 import workloads as WL

WEIGHT_RTOL = 1e-5


def build_both(net, oracle_mod, nc_mod, B=0, flags=0, finalize=True):
    o = oracle_mod.Oracle(dt_ms=net.dt_ms, block_size=B)
    WL.run(net, o, finalize=finalize)
    g = nc_mod.NC(dt_ms=net.dt_ms, block_size=B, flags=flags)
    WL.run(net, g, finalize=finalize)
    return o, g


def weight_scale(net):
    return max(abs(p.weight[0]) + p.weight[1] for p in net.projections)


def compare_connections(gc, oc, scale, what=""):
    """gc: dict from NC.read_connections, oc: dict from Oracle.connections.  Returns the mismatch report."""
    n = oc["n"]
    assert gc["n"] == n, (what, gc["n"], n)
    assert np.array_equal(gc["source"], oc["source"]), f"{what}: sources differ"
    assert np.array_equal(gc["target"], oc["target"]), f"{what}: targets differ"
    if "perm" in oc:
        assert np.array_equal(gc["perm"], oc["perm"]), f"{what}: permutation differs"
    # weights: |dw| <= 1e-5 * max(|w|, weight scale of the network)
    dw = np.abs(gc["weight"].astype(np.float64) - oc["weight"].astype(np.float64))
    tol = WEIGHT_RTOL * np.maximum(np.abs(oc["weight"].astype(np.float64)), scale)
    assert np.all(dw <= tol), f"{what}: weight error {dw.max()} (rel {np.max(dw / tol) * WEIGHT_RTOL:.3g})"
    # delays
    dd = gc["delay"].astype(np.int64) - oc["delay"].astype(np.int64)
    bad = np.flatnonzero(dd)
    report = {"n": int(n), "delay_mismatches": int(bad.size), "max_weight_rel_err": float(np.max(dw / np.maximum(np.abs(oc["weight"]), scale))) if n else 0.0}
    if bad.size:
        assert np.all(np.abs(dd[bad]) == 1), f"{what}: a delay differs by more than one step"
        assert np.all(oc["boundary"][bad] == 1), f"{what}: {bad.size} delay mismatches away from a rounding boundary (first at {bad[0]})"
        assert bad.size <= math.ceil(1e-7 * n), f"{what}: {bad.size} boundary mismatches > 1e-7 of {n}"
    return report


def compare_index(gi, oi, what=""):
    for k in ("n_nodes", "total_groups"):
        assert gi[k] == oi[k], (what, k, gi[k], oi[k])
    for k in ("src_offsets", "group_count", "group_ptr", "group_start", "group_delay"):
        assert np.array_equal(gi[k], oi[k]), f"{what}: {k} differs"


def full_parity(net, oracle_mod, nc_mod, B=0, flags=0):
    o, g = build_both(net, oracle_mod, nc_mod, B=B, flags=flags)
    scale = weight_scale(net)
    rep = compare_connections(g.read_connections(sorted=False), o.connections(sorted=False), scale, net.name + " creation order")
    ou, os_ = o.connections(sorted=False), o.connections(sorted=True)
    gs = g.read_connections(sorted=True)
    if rep["delay_mismatches"] == 0:
        rep_s = compare_connections(gs, os_, scale, net.name + " sorted")
        compare_index(g.read_index(), o.index(), net.name)
    else:
        # a boundary delay moved by one step: the GPU order is the stable sort of ITS OWN (source, delay)
        gu = g.read_connections(sorted=False)
        key = (gu["source"].astype(np.uint64) << np.uint64(16)) | gu["delay"].astype(np.uint64)
        perm = np.argsort(key, kind="stable").astype(np.uint32)
        assert np.array_equal(gs["perm"], perm)
        rep_s = rep
    for kind in (0, 1):
        gd, gm = g.read_degree_histogram(kind)
        od, om = o.degree_histogram(kind)
        assert np.array_equal(gd, od) and gm == om, f"{net.name}: degree histogram kind {kind}"
    assert g.stats()["n_blocks"] == o.num_blocks(), "Eq. 1 block count"
    g.close()
    return rep, rep_s
