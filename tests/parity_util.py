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


def weight_scale(net, o=None, perm=None):
    """Tolerance floor of the weight comparison.  With the oracle `o` the recipe was replayed on: one value per
    connection, the scale |mean| + sd of the synapse's OWN projection (in creation order, or gathered by `perm` for
    the organised view).  Without it: the largest projection scale of the network (callers that only hold a recipe)."""
    per_proj = [abs(p.weight[0]) + p.weight[1] for p in net.projections]
    if o is None:
        return max(per_proj)
    return scale_per_connection(per_proj, o, perm)


def scale_per_connection(per_proj, o, perm=None):
    starts = o.projection_starts()
    assert starts.size == len(per_proj) + 1, (starts.size, len(per_proj))
    arr = np.repeat(np.asarray(per_proj, dtype=np.float32), np.diff(starts))
    return arr if perm is None else arr[perm]


CHUNK = 1 << 25


def compare_connections(gc, oc, scale, what="", max_mismatch=None):
    """gc: dict from NC.read_connections, oc: dict from Oracle.connections.  `scale`: a number or one value per
    connection (weight_scale).  Sources, targets, permutation bit-exact; |dw| <= 1e-5 * max(|w|, scale); delays equal
    except for at most ceil(1e-7 n) synapses that the oracle flags as rounding boundaries (reading D8), each off by
    one step.  Every mismatch is counted; returns the report."""
    n = oc["n"]
    assert gc["n"] == n, (what, gc["n"], n)
    per_conn = isinstance(scale, np.ndarray)
    if per_conn:
        assert scale.shape == (n,)
    n_bad, max_rel = 0, 0.0
    for a in range(0, n, CHUNK):
        sl = slice(a, min(n, a + CHUNK))
        assert np.array_equal(gc["source"][sl], oc["source"][sl]), f"{what}: sources differ"
        assert np.array_equal(gc["target"][sl], oc["target"][sl]), f"{what}: targets differ"
        if "perm" in oc:
            assert np.array_equal(gc["perm"][sl], oc["perm"][sl]), f"{what}: permutation differs"
        ow = oc["weight"][sl].astype(np.float64)
        dw = np.abs(gc["weight"][sl].astype(np.float64) - ow)
        ref = np.maximum(np.abs(ow), scale[sl] if per_conn else scale)
        rel = float(np.max(dw / ref)) if dw.size else 0.0
        assert rel <= WEIGHT_RTOL, f"{what}: weight error {rel:.3g} relative to the projection scale (abs {dw.max():.3g})"
        max_rel = max(max_rel, rel)
        dd = gc["delay"][sl].astype(np.int32) - oc["delay"][sl].astype(np.int32)
        bad = np.flatnonzero(dd)
        if bad.size:
            assert np.all(np.abs(dd[bad]) == 1), f"{what}: a delay differs by more than one step"
            assert np.all(oc["boundary"][sl][bad] == 1), \
                f"{what}: {bad.size} delay mismatches away from a rounding boundary (first at {a + bad[0]})"
            n_bad += int(bad.size)
    allowed = math.ceil(1e-7 * n) if max_mismatch is None else max_mismatch  # a chunk of a larger comparison passes its own
    assert n_bad <= allowed, f"{what}: {n_bad} boundary mismatches > {allowed} (1e-7 of the connections compared)"
    return {"n": int(n), "delay_mismatches": n_bad, "max_weight_rel_err": max_rel}


def compare_sorted(g, o, net, what=""):
    """Organised view of the CUDA path against the oracle's, weight floor = the synapse's own projection scale."""
    os_ = o.connections(sorted=True)
    return compare_connections(g.read_connections(sorted=True), os_, weight_scale(net, o, os_["perm"]), what)


def compare_index(gi, oi, what=""):
    for k in ("n_nodes", "total_groups"):
        assert gi[k] == oi[k], (what, k, gi[k], oi[k])
    for k in ("src_offsets", "group_count", "group_ptr", "group_start", "group_delay"):
        assert np.array_equal(gi[k], oi[k]), f"{what}: {k} differs"


def full_parity(net, oracle_mod, nc_mod, B=0, flags=0):
    o, g = build_both(net, oracle_mod, nc_mod, B=B, flags=flags)
    rep = compare_connections(g.read_connections(sorted=False), o.connections(sorted=False), weight_scale(net, o),
                              net.name + " creation order")
    os_ = o.connections(sorted=True)
    gs = g.read_connections(sorted=True)
    if rep["delay_mismatches"] == 0:
        rep_s = compare_connections(gs, os_, weight_scale(net, o, os_["perm"]), net.name + " sorted")
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
