"""GPU parity tests proper: the CUDA path, called through the C ABI, against the CPU oracle on the same
seeded recipes -- element by element at sizes the oracle finishes in seconds (several sort tiles plus a
ragged tail), edge cases, and device self-tests of the RNG and of the fp32 fast path."""
import math

import numpy as np
import pytest

from paper_2306_09855_b200 import workloads as WL
from tests import parity_util as PU

pytestmark = pytest.mark.gpu
INF = math.inf
W = (20.0, 2.0, 0.0, INF)
D = (1.5, 0.75, 0.1, INF)


@pytest.fixture(scope="module")
def nc_mod():
    from paper_2306_09855_b200 import binding, build
    build.build()
    return binding


def test_device_philox_matches_known_answers_and_oracle(nc_mod, oracle_mod):
    g = nc_mod.NC()
    ctr = np.array([[0, 0, 0, 0], [0xffffffff] * 4, [0x243f6a88, 0x85a308d3, 0x13198a2e, 0x03707344]], dtype=np.uint32)
    key = np.array([[0, 0], [0xffffffff] * 2, [0xa4093822, 0x299f31d0]], dtype=np.uint32)
    out = g.selftest_philox(ctr, key)
    want = np.array([[0x6627e8d5, 0xe169c58d, 0xbc57ac4c, 0x9b00dbd8], [0x408f276d, 0x41c83b0e, 0xa20bc7c6, 0x6d5451fd],
                     [0xd16cfe09, 0x94fdcceb, 0x5001e420, 0x24126ea1]], dtype=np.uint32)
    assert np.array_equal(out, want)
    rng = np.random.default_rng(1)
    ctr = rng.integers(0, 2**32, size=(2000, 4), dtype=np.uint64).astype(np.uint32)
    key = rng.integers(0, 2**32, size=(2000, 2), dtype=np.uint64).astype(np.uint32)
    out = g.selftest_philox(ctr, key)
    ref = np.array([oracle_mod.philox4x32_10(c.tolist(), k.tolist()) for c, k in zip(ctr, key)], dtype=np.uint32)
    assert np.array_equal(out, ref)
    g.close()


def test_fastpath_error_is_inside_the_guard_band(nc_mod):
    """Exhaustive over all 2^24 u1 and all 2^24 u2 on the device: the special-function fast path of the
    radius and of sin/cos stays within a quarter of the error bound the delay guard band assumes (DESIGN.md
    'delay fast path'), and the radius is accurate enough in absolute terms for the 1e-5 weight tolerance
    (weight error <= sd_w (|dr| + r |dcos|), tolerance >= 1e-5 sd_w)."""
    g = nc_mod.NC()
    ratio_r, ratio_sin, ratio_cos, abs_r = g.selftest_fastpath()
    g.close()
    print(f"fast path: worst error/bound: r {ratio_r:.3f}, sin {ratio_sin:.3f}, cos {ratio_cos:.3f}; max abs err r {abs_r:.3e}")
    assert ratio_r < 0.25 and ratio_sin < 0.25 and ratio_cos < 0.25
    assert abs_r < 4e-6


@pytest.mark.parametrize("B", [0, 10, 64, 1000])
def test_config0_tiny_full_parity(nc_mod, oracle_mod, B):
    rep, rep_s = PU.full_parity(WL.config0_tiny(), oracle_mod, nc_mod, B=B)
    assert rep["n"] == 1000 and rep["delay_mismatches"] == 0


@pytest.mark.parametrize("rule,scale", [("one_to_one", 1.0), ("all_to_all", 0.15), ("fixed_indegree", 0.3),
                                        ("fixed_outdegree", 0.25), ("fixed_total_number", 0.3),
                                        ("pairwise_bernoulli", 0.4),
                                        # BASELINE.json configs[1] at its full size, every connection against the oracle:
                                        # 10^8, 2 * 10^7 and 4 * 10^7 connections
                                        ("all_to_all", 1.0), ("fixed_outdegree", 1.0), ("fixed_total_number", 1.0)])
def test_config1_rule_sweep_parity(nc_mod, oracle_mod, rule, scale):
    net = WL.config1_rule(rule, scale=scale)
    rep, _ = PU.full_parity(net, oracle_mod, nc_mod)
    print(net.name, rep)
    assert rep["n"] > 5000


def test_config1_exact_fp64_flag_gives_same_delays(nc_mod, oracle_mod):
    net = WL.config1_rule("fixed_total_number", scale=0.2)
    rep, _ = PU.full_parity(net, oracle_mod, nc_mod, flags=nc_mod.FLAG_EXACT_FP64)
    assert rep["delay_mismatches"] == 0


def test_microcircuit_scaled_parity(nc_mod, oracle_mod):
    """configs[2] at 10 % of the populations (same probabilities): 55 projections, ~3e6 synapses, I and E delays."""
    net = WL.config2_microcircuit(scale=0.1)
    rep, _ = PU.full_parity(net, oracle_mod, nc_mod)
    print(net.name, rep)
    assert len(net.projections) >= 50 and rep["n"] > 2_000_000


def test_sort_pairs_variant_parity(nc_mod, oracle_mod):
    """NC_FLAG_SORT_PAIRS: (key, position) pairs + gather by the permutation instead of carrying the connection."""
    for net in (WL.config2_microcircuit(scale=0.06), WL.config1_rule("fixed_indegree", scale=0.2)):
        rep, _ = PU.full_parity(net, oracle_mod, nc_mod, flags=nc_mod.FLAG_SORT_PAIRS)
        assert rep["n"] > 300_000


def test_onesweep_lookback_variant_parity(nc_mod, oracle_mod):
    """NC_FLAG_SORT_ONESWEEP: whole connections carried through single-pass digit sweeps chained by decoupled
    look-back (the alternative to the default count / scan / scatter kernels per pass)."""
    for net in (WL.config2_microcircuit(scale=0.06), WL.config1_rule("fixed_indegree", scale=0.2)):
        rep, _ = PU.full_parity(net, oracle_mod, nc_mod, flags=nc_mod.FLAG_SORT_ONESWEEP)
        assert rep["n"] > 300_000


def test_bulk_fed_persistent_variant_parity(nc_mod, oracle_mod, monkeypatch):
    """NC_FLAG_SORT_BULK: every digit pass as a persistent kernel fed by cp.async.bulk (nc_sort_bulk.cuh): first pass from
    the SoA slices of the storage blocks (B a multiple of the tile) or through the default kernel (odd B), middle
    passes with one bulk store per digit run, last pass into the final arrays; ragged last tile; several blocks.  Ranks
    from ballots (the default) and from returning shared atomics (NC_ATOMIC_RANK=1, opt-in)."""
    for atomic in (None, "1"):
        if atomic is None:
            monkeypatch.delenv("NC_ATOMIC_RANK", raising=False)
        else:
            monkeypatch.setenv("NC_ATOMIC_RANK", atomic)
        for net, B in ((WL.config2_microcircuit(scale=0.06), 0), (WL.config1_rule("fixed_indegree", scale=0.2), 1 << 16),
                       (WL.config1_rule("fixed_total_number", scale=0.05), 100_003), (WL.config0_tiny(), 64)):
            rep, _ = PU.full_parity(net, oracle_mod, nc_mod, flags=nc_mod.FLAG_SORT_BULK, B=B)
            assert rep["n"] >= 1000
    monkeypatch.delenv("NC_ATOMIC_RANK", raising=False)


def test_bucket_first_variant_parity(nc_mod, oracle_mod, monkeypatch):
    """NC_FLAG_SORT_BUCKETS (nc_sort_msd.cuh): one pass into <= 256 buckets of consecutive sources, then every bucket sorted on
    its own with its intermediate records in an L2-resident slot.  Same connections, permutation and index as the oracle:
    several storage blocks, odd B (scalar first pass), tiny networks (most buckets empty, N < 256), one, two and three
    in-bucket passes, the persistent kernel and the per-bucket launches over 1 - 4 CUDA streams, one bucket that holds
    everything."""
    for net, B in ((WL.config2_microcircuit(scale=0.06), 0), (WL.config1_rule("fixed_indegree", scale=0.2), 1 << 16),
                   (WL.config1_rule("fixed_total_number", scale=0.05), 100_003), (WL.config0_tiny(), 64),
                   (WL.config1_rule("pairwise_bernoulli", scale=0.1), 0)):
        for lanes in (None, "1", "2", "3", "4"):  # None: the persistent kernel where it applies (two in-bucket passes)
            if lanes is None:
                monkeypatch.delenv("NC_BUCKET_LANES", raising=False)
            else:
                monkeypatch.setenv("NC_BUCKET_LANES", lanes)
            rep, _ = PU.full_parity(net, oracle_mod, nc_mod, flags=nc_mod.FLAG_SORT_BUCKETS, B=B)
            assert rep["n"] >= 1000
    monkeypatch.delenv("NC_BUCKET_LANES")
    monkeypatch.setenv("NC_ATOMIC_RANK", "1")  # opt-in: ranks from returning shared atomics in the persistent bucket kernel
    rep, _ = PU.full_parity(WL.config2_microcircuit(scale=0.06), oracle_mod, nc_mod, flags=nc_mod.FLAG_SORT_BUCKETS)
    assert rep["n"] >= 1000
    monkeypatch.delenv("NC_ATOMIC_RANK")
    # 16 nodes, delays up to 15 steps: 4 delay bits + 1 -> one in-bucket pass
    net = WL.Network("narrow", [16])
    net.projections = [WL.Projection(0, 0, "fixed_total_number", degree_or_total=100_000, weight=W,
                                     delay_ms=(0.5, 0.3, 0.1, 1.5), seed=8)]
    o, g = PU.build_both(net, oracle_mod, nc_mod, flags=nc_mod.FLAG_SORT_BUCKETS)
    assert g.stats()["sort_passes"] == 2
    g.close(); o.close()
    PU.full_parity(net, oracle_mod, nc_mod, flags=nc_mod.FLAG_SORT_BUCKETS)
    # 3,000,000 nodes x delays up to 2^9 steps: 14 source bits left in a bucket + 10 delay bits -> three in-bucket passes
    net = WL.Network("wide", [3_000_000])
    net.projections = [WL.Projection(0, 0, "fixed_total_number", degree_or_total=1_500_000, weight=W,
                                     delay_ms=(20.0, 15.0, 0.1, 51.0), seed=11)]
    o, g = PU.build_both(net, oracle_mod, nc_mod, flags=nc_mod.FLAG_SORT_BUCKETS)
    assert g.stats()["sort_passes"] == 4
    g.close(); o.close()
    PU.full_parity(net, oracle_mod, nc_mod, flags=nc_mod.FLAG_SORT_BUCKETS)
    # every connection from 3 neighbouring sources of 100,000: one bucket holds everything
    net = WL.Network("one_bucket", [100_000])
    net.projections = [WL.Projection(0, 0, "fixed_total_number", degree_or_total=2000, weight=W, delay_ms=(1.5, 0.75, 0.1, 4.0), seed=3)]
    o = oracle_mod.Oracle(dt_ms=net.dt_ms)
    g = nc_mod.NC(dt_ms=net.dt_ms, flags=nc_mod.FLAG_SORT_BUCKETS)
    for b in (o, g):
        b.create_population(100_000)
        b.connect((0, 100_000), (0, 100_000), WL.RULE_IDS["fixed_total_number"], degree_or_total=2000, weight=(1.0, 0.0, 0.0, float("inf")),
                  delay_ms=(1.5, 0.75, 0.1, 4.0), seed=3)
        b.connect((5000, 3), (0, 100_000), WL.RULE_IDS["all_to_all"], weight=(1.0, 0.0, 0.0, float("inf")),
                  delay_ms=(1.5, 0.75, 0.1, 4.0), seed=4)
        b.finalize()
    PU.compare_connections(g.read_connections(sorted=True), o.connections(sorted=True), 1.0, "one bucket")
    PU.compare_index(g.read_index(), o.index(), "one bucket")
    g.close(); o.close()


def test_single_pass_key(nc_mod, oracle_mod):
    """<= 8 key bits: one digit pass that is both the first and the last (storage blocks -> final arrays)."""
    net = WL.Network("narrow", [16])
    net.projections = [WL.Projection(0, 0, "fixed_total_number", degree_or_total=100_000, weight=W,
                                     delay_ms=(0.5, 0.3, 0.1, 1.5), seed=8)]
    o, g = PU.build_both(net, oracle_mod, nc_mod)
    assert g.stats()["sort_passes"] == 1
    g.close()
    PU.full_parity(net, oracle_mod, nc_mod)
    PU.full_parity(net, oracle_mod, nc_mod, flags=nc_mod.FLAG_SORT_PAIRS)
    PU.full_parity(net, oracle_mod, nc_mod, flags=nc_mod.FLAG_SORT_ONESWEEP)
    PU.full_parity(net, oracle_mod, nc_mod, flags=nc_mod.FLAG_SORT_BULK)


def test_block_sizes_paper_default_and_odd(nc_mod, oracle_mod):
    """B = 10^7 (the paper's default, not a power of two -> magic division) and an odd B (scalar stores)."""
    net = WL.config3_large_indegree(scale=0.02)  # 1600+400 nodes, K = 160 / 40 -> 400k synapses
    for B in (10_000_000, 100_003, 4096):
        rep, _ = PU.full_parity(net, oracle_mod, nc_mod, B=B)
        assert rep["n"] == 2000 * 200


def test_bernoulli_and_outdegree_mix_scaled_c4(nc_mod, oracle_mod):
    net = WL.config4_large_bernoulli(scale=0.01)  # 1600 + 400 nodes: 4e6 trials, ~1e5 accepted, + K = 5 out-degree
    rep, _ = PU.full_parity(net, oracle_mod, nc_mod)
    assert rep["n"] > 90_000


def test_edge_cases(nc_mod, oracle_mod):
    # empty network
    g = nc_mod.NC()
    g.create_population(5)
    g.finalize()
    idx = g.read_index()
    assert idx["total_groups"] == 0 and idx["src_offsets"].tolist() == [0] * 6 and idx["group_ptr"].tolist() == [0] * 6
    assert g.read_connections(sorted=True)["n"] == 0
    g.close()
    # sources with no outgoing connection at both ends and in the middle; constant weight/delay; p = 0 and 1
    net = WL.Network("edges", [7, 50, 9, 30, 11])
    net.projections = [
        WL.Projection(1, 3, "pairwise_bernoulli", p=1.0, weight=W, delay_ms=D, seed=3),
        WL.Projection(3, 1, "pairwise_bernoulli", p=0.0, weight=W, delay_ms=D, seed=3),
        WL.Projection(3, 3, "one_to_one", weight=(2.5, 0.0, -INF, INF), delay_ms=(0.25, 0.0, -INF, INF), seed=3),
        WL.Projection(3, 0, "fixed_indegree", degree_or_total=0, weight=W, delay_ms=D, seed=3),
        WL.Projection(1, 1, "fixed_total_number", degree_or_total=1, weight=W, delay_ms=D, seed=3),
        WL.Projection(1, 3, "all_to_all", weight=(-1.0, 3.0, -2.0, 0.0), delay_ms=(1.0, 5.0, 0.1, 3.0), seed=4),
    ]
    rep, _ = PU.full_parity(net, oracle_mod, nc_mod, B=64)
    assert rep["n"] == 50 * 30 + 30 + 1 + 50 * 30
    # a single source with every connection (one huge group run) and delay bound at the u16 limit
    net2 = WL.Network("one_source", [1, 20000])
    net2.projections = [WL.Projection(0, 1, "all_to_all", weight=W, delay_ms=(6553.5, 0.0, -INF, INF), seed=1),
                        WL.Projection(0, 1, "fixed_outdegree", degree_or_total=30000, weight=W, delay_ms=D, seed=1)]
    rep2, _ = PU.full_parity(net2, oracle_mod, nc_mod)
    assert rep2["n"] == 50000


def test_wide_key_uses_64_bit_sort(nc_mod, oracle_mod):
    """2^17 nodes and delays up to 65535 steps -> 17 + 16 = 33 key bits -> the u64 instantiation."""
    net = WL.Network("wide", [131072])
    net.projections = [WL.Projection(0, 0, "fixed_total_number", degree_or_total=300_000, weight=W,
                                     delay_ms=(3000.0, 1500.0, 0.1, 6553.5), seed=8)]
    o, g = PU.build_both(net, oracle_mod, nc_mod)
    assert g.stats()["key_bits"] == 33 and g.stats()["sort_passes"] == 5
    PU.compare_sorted(g, o, net, "wide")
    PU.compare_index(g.read_index(), o.index(), "wide")
    g.close()


def test_error_codes_match_oracle(nc_mod, oracle_mod):
    g = nc_mod.NC()
    o = oracle_mod.Oracle(dt_ms=0.1)
    for b in (g, o):
        b.create_population(10)
        b.create_population(20)
    ok = dict(weight=W, delay_ms=D, seed=1)
    cases = [
        ((0, 10), (10, 20), 0, {}),                            # one_to_one size mismatch
        ((25, 10), (10, 20), 1, {}),                           # outside created nodes
        ((0, 0), (10, 20), 1, {}),                             # empty range
        ((0, 10), (10, 20), 5, dict(p=1.5)),
        ((0, 10), (10, 20), 9, {}),
        ((0, 10), (10, 20), 4, dict(degree_or_total=2**32)),
        ((0, 10), (10, 20), 2, dict(degree_or_total=2**31)),
    ]
    for src, tgt, rule, extra in cases:
        assert g.connect_rc(src, tgt, rule, **extra, **ok) == o.connect_rc(src, tgt, rule, **extra, **ok) != 0
    bad_w = dict(weight=(1, -1, -INF, INF), delay_ms=D, seed=1)
    assert g.connect_rc((0, 10), (10, 20), 1, **bad_w) == o.connect_rc((0, 10), (10, 20), 1, **bad_w) == nc_mod.ERR_INVALID_ARG
    big_d = dict(weight=W, delay_ms=(7000.0, 0.0, -INF, INF), seed=1)
    assert g.connect_rc((0, 10), (10, 20), 1, **big_d) == o.connect_rc((0, 10), (10, 20), 1, **big_d) == nc_mod.ERR_CAPACITY
    assert g.num_connections() == 0
    g.connect((0, 10), (10, 20), 4, degree_or_total=5, **ok)  # projection id 0: failures consumed none
    o.connect((0, 10), (10, 20), 4, degree_or_total=5, **ok)
    assert np.array_equal(g.read_connections()["source"], o.connections()["source"])
    with pytest.raises(nc_mod.NCError):
        g.read_connections(sorted=True)
    g.finalize()
    assert g.connect_rc((0, 10), (10, 20), 1, **ok) == nc_mod.ERR_STATE
    with pytest.raises(nc_mod.NCError):
        g.finalize()
    g.close()


def test_default_cuda_allocator_path(nc_mod, oracle_mod):
    """mem.alloc == NULL -> cudaMalloc/cudaFree inside the library."""
    net = WL.config0_tiny()
    o = oracle_mod.Oracle(dt_ms=0.1)
    WL.run(net, o)
    g = nc_mod.NC(use_torch_allocator=False)
    WL.run(net, g)
    PU.compare_sorted(g, o, net, "cudaMalloc")
    g.close()


def _report(name, rep):
    """The mismatch count goes to the log whatever the capture settings are: printed, raised as a warning (pytest's
    summary lists it) and written beside the other artefacts of a GPU run."""
    import json, os, warnings
    msg = f"parity report {name}: {json.dumps(rep)}"
    print(msg)
    warnings.warn(msg)
    try:
        os.makedirs("gpurun_out", exist_ok=True)
        with open(os.path.join("gpurun_out", f"parity_{name}.json"), "w") as f:
            json.dump(rep, f)
    except OSError:
        pass


def test_full_size_microcircuit_every_connection_against_oracle(nc_mod, oracle_mod):
    """configs[2] at FULL size (77,169 nodes, 298,880,970 connections), built exactly as bench.py builds it, and
    built by the oracle too (about two minutes and 12 GB on the host): EVERY connection is compared -- creation-order
    sources and targets bit-exact, weights within 1e-5 of the synapse's own projection scale, delays with every
    mismatch counted, allowed only where the oracle flags a rounding boundary (reading D8) and at most
    ceil(1e-7 n) = 30 of them; then the permutation, the organised arrays and all five index arrays against
    oc_finalize.  The counts are reported."""
    net = WL.config2_microcircuit()
    g = nc_mod.NC(dt_ms=net.dt_ms)
    WL.run(net, g)
    n = g.num_connections()
    assert n == 298_880_970 and g.num_nodes() == 77_169
    st = g.stats()
    assert st["key_bits"] == 23
    o = oracle_mod.Oracle(dt_ms=net.dt_ms)
    WL.run(net, o)
    assert o.num_connections() == n
    chunk = 1 << 26
    total = {"n": n, "delay_mismatches": 0, "max_weight_rel_err": 0.0, "boundary_flags": 0}

    def compare_view(sorted_view):
        ov = o.connections(sorted=sorted_view, copy=False)
        scale_proj = np.asarray([abs(p.weight[0]) + p.weight[1] for p in net.projections], dtype=np.float32)
        starts = o.projection_starts()
        bad = 0
        for a in range(0, n, chunk):
            c = min(chunk, n - a)
            gv = g.read_connections(sorted=sorted_view, first=a, count=c)
            osl = {k: (v[a:a + c] if isinstance(v, np.ndarray) else v) for k, v in ov.items()}
            osl["n"] = c
            pos = osl["perm"].astype(np.int64) if sorted_view else np.arange(a, a + c, dtype=np.int64)
            scale = scale_proj[np.searchsorted(starts, pos, side="right") - 1]
            rep = PU.compare_connections(gv, osl, scale, f"c2 full, {'organised' if sorted_view else 'creation'} order, "
                                         f"chunk at {a}", max_mismatch=30)
            bad += rep["delay_mismatches"]
            total["max_weight_rel_err"] = max(total["max_weight_rel_err"], rep["max_weight_rel_err"])
        return bad, int(ov["boundary"].sum(dtype=np.int64))

    total["delay_mismatches"], total["boundary_flags"] = compare_view(False)
    assert total["delay_mismatches"] <= math.ceil(1e-7 * n) == 30
    if total["delay_mismatches"] == 0:
        bad_s, _ = compare_view(True)
        assert bad_s == 0
        PU.compare_index(g.read_index(), o.index(), "c2 full")
        total["organised_and_index_vs_oracle"] = "bit-exact"
    else:
        # a boundary delay moved by one step: the device's order is the stable sort of ITS OWN (source, delay)
        gu = g.read_connections(sorted=False, fields=("source", "delay"))
        key = (gu["source"].astype(np.uint64) << np.uint64(16)) | gu["delay"].astype(np.uint64)
        gs = g.read_connections(sorted=True, fields=("perm",))
        assert np.array_equal(gs["perm"], np.argsort(key, kind="stable").astype(np.uint32))
        total["organised_and_index_vs_oracle"] = "own keys (a boundary delay differs)"
    for kind in (0, 1):
        gd, gm = g.read_degree_histogram(kind)
        od, om = o.degree_histogram(kind)
        assert np.array_equal(gd, od) and gm == om
    _report("c2_full", total)
    g.close()
    o.close()


def _check_organised_chunked(g, n, n_nodes, chunk=40_000_000):
    """Readings D10/D11 checked on the device's own arrays at any size, a chunk of the sorted order at a time:
    perm is a permutation, keys ascend, ties keep creation order, source and delay are the gathered creation-order
    values, and every index array equals its definition."""
    u = g.read_connections(sorted=False, fields=("source", "delay"))
    seen = np.zeros(n, dtype=bool)
    out_deg = np.zeros(n_nodes, dtype=np.int64)
    gcount = np.zeros(n_nodes, dtype=np.int64)
    heads, head_delay = [], []
    prev_key, prev_perm = None, None
    for j0 in range(0, n, chunk):
        c = min(chunk, n - j0)
        s = g.read_connections(sorted=True, first=j0, count=c, fields=("source", "delay", "perm"))
        perm = s["perm"]
        assert not seen[perm].any(), "perm repeats a position"
        seen[perm] = True
        assert np.array_equal(u["source"][perm], s["source"]) and np.array_equal(u["delay"][perm], s["delay"])
        key = (s["source"].astype(np.uint64) << np.uint64(16)) | s["delay"].astype(np.uint64)
        if prev_key is not None:
            key = np.concatenate([[prev_key], key])
            perm = np.concatenate([[prev_perm], perm])
        dk = key[1:] != key[:-1]
        assert np.all(key[1:] >= key[:-1]), "not sorted by (source, delay)"
        assert np.all(dk | (perm[1:] > perm[:-1])), "ties are not in creation order"
        h = np.flatnonzero(dk) + (j0 if prev_key is not None else j0 + 1)
        if prev_key is None:
            h = np.concatenate([[0], h])
        heads.append(h.astype(np.uint32))
        head_delay.append(s["delay"][h - j0])
        out_deg += np.bincount(s["source"], minlength=n_nodes)
        gcount += np.bincount(s["source"][h - j0], minlength=n_nodes)
        prev_key, prev_perm = key[-1], perm[-1]
    assert seen.all(), "perm is not a permutation"
    idx = g.read_index()
    heads = np.concatenate(heads)
    assert idx["total_groups"] == heads.size
    assert np.array_equal(idx["group_start"], heads) and np.array_equal(idx["group_delay"], np.concatenate(head_delay))
    assert np.array_equal(idx["src_offsets"], np.concatenate([[0], np.cumsum(out_deg)]).astype(np.uint32))
    assert np.array_equal(idx["group_count"], gcount.astype(np.uint32))
    assert np.array_equal(idx["group_ptr"], np.concatenate([[0], np.cumsum(gcount)]).astype(np.uint32))


def _check_sampled_synapses(g, net, firsts, oracle_mod, starts, stride=16, chunk=1 << 26):
    """Every `stride`-th creation position of every projection whose i_newconns is the position inside the projection
    (all rules but pairwise_bernoulli), against the oracle's per-synapse function: sources and targets bit-exact,
    weights within 1e-5 of the projection's own scale, delay mismatches only on flagged boundaries, counted."""
    n = int(starts[-1])
    checked = mism = 0
    max_rel = 0.0
    for pj, pr in enumerate(net.projections):
        if pr.rule == "pairwise_bernoulli":
            continue
        p0, p1 = int(starts[pj]), int(starts[pj + 1])
        scale = abs(pr.weight[0]) + pr.weight[1]
        for a in range(p0, p1, chunk):
            c = min(chunk, p1 - a)
            got = g.read_connections(sorted=False, first=a, count=c)
            sel = np.unique(np.concatenate([np.arange(0, c, stride), [c - 1]]))
            want = oracle_mod.eval_synapses((firsts[pr.src_pop], net.populations[pr.src_pop]),
                                            (firsts[pr.tgt_pop], net.populations[pr.tgt_pop]), WL.RULE_IDS[pr.rule],
                                            pr.degree_or_total, pr.p, pr.weight, pr.delay_ms, pr.seed, pj, net.dt_ms,
                                            (a - p0) + sel)
            assert np.array_equal(got["source"][sel], want["source"]) and np.array_equal(got["target"][sel], want["target"]), pj
            ow = want["weight"].astype(np.float64)
            rel = np.abs(got["weight"][sel].astype(np.float64) - ow) / np.maximum(np.abs(ow), scale)
            assert rel.max() <= PU.WEIGHT_RTOL, (pj, rel.max())
            max_rel = max(max_rel, float(rel.max()))
            dd = got["delay"][sel].astype(np.int32) - want["delay"].astype(np.int32)
            bad = np.flatnonzero(dd)
            assert np.all(np.abs(dd[bad]) == 1) and np.all(want["boundary"][bad] == 1), pj
            mism += bad.size
            checked += sel.size
    assert mism <= math.ceil(1e-7 * checked)
    return {"checked": int(checked), "of": n, "delay_mismatches": int(mism), "max_weight_rel_err": max_rel}


def test_full_size_config3_large_indegree(nc_mod, oracle_mod):
    """configs[3]: 100,000 nodes, 10^9 connections (fixed_indegree 8000 / 2000)."""
    net = WL.config3_large_indegree()
    g = nc_mod.NC(dt_ms=net.dt_ms)
    firsts = WL.run(net, g)
    n = g.num_connections()
    assert n == 1_000_000_000
    sizes = np.array([net.populations[p.tgt_pop] * p.degree_or_total for p in net.projections], dtype=np.int64)
    starts = np.concatenate([[0], np.cumsum(sizes)])
    rep = _check_sampled_synapses(g, net, firsts, oracle_mod, starts, stride=16)
    assert rep["checked"] >= 60_000_000
    _report("c3_sampled", rep)
    deg, mx = g.read_degree_histogram(0)
    assert np.all(deg == 10_000) and mx == 10_000  # exact in-degree K_E + K_I per target (Eq. 11)
    _check_organised_chunked(g, n, net.n_nodes)
    g.close()


def test_full_size_config4_large_bernoulli(nc_mod, oracle_mod):
    """configs[4]: 200,000 nodes, 4 x pairwise_bernoulli p = 0.025 over 4e10 pairs + fixed_outdegree K = 500.
    Bernoulli projections: the count is within 5 sigma of the binomial, pairs ascend in q (D4), every sampled pair
    is one the oracle's trial stream accepts and carries the oracle's weight and delay for that q, and the accepted
    set inside windows of 200,000 pairs (the first and last pairs of every projection, both sides of q = 2^32, 2^33, 2^34)
    is exactly the oracle's."""
    net = WL.config4_large_bernoulli()
    g = nc_mod.NC(dt_ms=net.dt_ms)
    firsts = [g.create_population(p) for p in net.populations]
    counts = []
    for pr in net.projections:
        before = g.num_connections()
        g.connect((firsts[pr.src_pop], net.populations[pr.src_pop]), (firsts[pr.tgt_pop], net.populations[pr.tgt_pop]),
                  WL.RULE_IDS[pr.rule], degree_or_total=pr.degree_or_total, p=pr.p, weight=pr.weight,
                  delay_ms=pr.delay_ms, seed=pr.seed)
        counts.append(g.num_connections() - before)
    g.finalize()
    n = g.num_connections()
    starts = np.concatenate([[0], np.cumsum(counts)]).astype(np.int64)
    bern_checked = bern_mism = 0
    win_count = win_pairs = win_accepted = 0
    for pj, pr in enumerate(net.projections):
        ns, nt = net.populations[pr.src_pop], net.populations[pr.tgt_pop]
        s0, t0 = firsts[pr.src_pop], firsts[pr.tgt_pop]
        if pr.rule != "pairwise_bernoulli":
            assert counts[pj] == ns * pr.degree_or_total
            continue
        T = oracle_mod.bernoulli_threshold(pr.p)
        pt = T / 2.0**32
        mean, sd = ns * nt * pt, math.sqrt(ns * nt * pt * (1 - pt))
        assert abs(counts[pj] - mean) < 5 * sd, (pj, counts[pj], mean, sd)
        # the head of the projection: exactly the oracle's accepted pairs among q < 200,000
        head = g.read_connections(sorted=False, first=int(starts[pj]), count=min(8000, counts[pj]))
        q = (head["source"].astype(np.int64) - s0) * nt + (head["target"].astype(np.int64) - t0)
        assert np.all(np.diff(q) > 0)
        want = [qq for qq in range(200_000) if oracle_mod.bernoulli_trial_word(pr.seed, pj, qq) < T]
        assert np.array_equal(q[q < 200_000], np.array(want, dtype=np.int64))
        # every 64th accepted pair of the projection, streamed: the pair index q rebuilt from (source, target) must
        # ascend, be one the oracle's trial stream accepts, and carry the oracle's weight and delay for that q
        # completeness, not only soundness: inside windows of 200,000 pairs -- the first pairs, both sides of q = 2^32, 2^33
        # and 2^34 (where the 64-bit counter path, the mask words and the tile counts change regime) and the last pairs of
        # the projection -- the device's accepted set must be EXACTLY the oracle's (a dropped pair fails here)
        n_pairs, WIN = ns * nt, 200_000
        wins = [0, n_pairs - WIN] + [c - WIN // 2 for c in (2**32, 2**33, 2**34) if c + WIN // 2 <= n_pairs]
        got_win = {w0: [] for w0 in wins}
        chunk = 1 << 26
        last_q = -1
        for a0 in range(int(starts[pj]), int(starts[pj + 1]), chunk):
            c = min(chunk, int(starts[pj + 1]) - a0)
            got = g.read_connections(sorted=False, first=a0, count=c)
            q = (got["source"].astype(np.int64) - s0) * nt + (got["target"].astype(np.int64) - t0)
            assert q[0] > last_q and np.all(np.diff(q) > 0) and q[-1] < ns * nt
            last_q = int(q[-1])
            for w0 in wins:
                lo, hi = np.searchsorted(q, [w0, w0 + WIN])
                if hi > lo:
                    got_win[w0].append(q[lo:hi].copy())
            sel = np.arange(0, c, 64)
            want = oracle_mod.eval_synapses((s0, ns), (t0, nt), WL.RULE_IDS[pr.rule], 0, pr.p, pr.weight, pr.delay_ms,
                                            pr.seed, pj, net.dt_ms, q[sel])
            assert np.all(want["accepted"] == 1), "a pair the oracle's trial stream rejects"
            assert np.array_equal(want["source"], got["source"][sel]) and np.array_equal(want["target"], got["target"][sel])
            ow = want["weight"].astype(np.float64)
            rel = np.abs(got["weight"][sel].astype(np.float64) - ow) / np.maximum(np.abs(ow), abs(pr.weight[0]) + pr.weight[1])
            assert rel.max() <= PU.WEIGHT_RTOL
            dd = got["delay"][sel].astype(np.int32) - want["delay"].astype(np.int32)
            bad = np.flatnonzero(dd)
            assert np.all(np.abs(dd[bad]) == 1) and np.all(want["boundary"][bad] == 1)
            bern_checked += sel.size
            bern_mism += bad.size
        for w0 in wins:
            idx = np.arange(w0, w0 + WIN, dtype=np.uint64)
            acc = oracle_mod.eval_synapses((s0, ns), (t0, nt), WL.RULE_IDS[pr.rule], 0, pr.p, pr.weight, pr.delay_ms, pr.seed,
                                           pj, net.dt_ms, idx)["accepted"]
            want_q = idx[acc == 1].astype(np.int64)
            have_q = np.concatenate(got_win[w0]) if got_win[w0] else np.zeros(0, np.int64)
            assert np.array_equal(have_q, want_q), f"projection {pj}: accepted pairs in [{w0}, {w0 + WIN}) differ from the oracle's"
            win_pairs += WIN
            win_accepted += int(want_q.size)
        win_count += len(wins)
    rep = _check_sampled_synapses(g, net, firsts, oracle_mod, starts, stride=4)  # the fixed_outdegree projection
    assert rep["checked"] >= 20_000_000
    _report("c4_sampled_outdegree", rep)
    assert bern_checked >= 15_000_000 and bern_mism <= math.ceil(1e-7 * bern_checked)
    _report("c4_sampled_bernoulli", {"checked": int(bern_checked), "delay_mismatches": int(bern_mism)})
    assert win_count >= 4 * 2 + 3 + 1 + 1  # head and tail of four projections; 2^32 in three of them, 2^33 and 2^34 in the largest
    _report("c4_bernoulli_exact_windows", {"windows": int(win_count), "pairs_tried": int(win_pairs),
                                           "accepted_in_windows": int(win_accepted), "set_differences": 0})
    _check_organised_chunked(g, n, net.n_nodes)
    g.close()


def test_explicit_node_arrays_parity(nc_mod, oracle_mod):
    """nc_connect_nodes: sources and/or targets given as arrays of node ids (unsorted, repeated ids,
    longer than a tile), every rule, mixed with range projections -- bit-exact against the oracle including the
    organised arrays and the index."""
    rng = np.random.default_rng(17)
    n_nodes = 3000
    src_ids = rng.choice(n_nodes, size=700, replace=False).astype(np.uint32)
    tgt_ids = rng.integers(0, n_nodes, size=900).astype(np.uint32)  # with repeats
    calls = [
        (src_ids, tgt_ids, "fixed_total_number", dict(degree_or_total=300_000)),
        ((100, 500), tgt_ids, "fixed_indegree", dict(degree_or_total=37)),
        (src_ids, (0, 3000), "fixed_outdegree", dict(degree_or_total=41)),
        (src_ids[:300], tgt_ids[:300], "one_to_one", {}),
        (src_ids[:64], tgt_ids[:100], "all_to_all", {}),
        (src_ids, tgt_ids, "pairwise_bernoulli", dict(p=0.05)),
        ((0, 3000), (0, 3000), "fixed_total_number", dict(degree_or_total=50_000)),
    ]
    o, g = oracle_mod.Oracle(dt_ms=0.1), nc_mod.NC(dt_ms=0.1)
    for b in (o, g):
        b.create_population(n_nodes)
        for s, t, rule, kw in calls:
            b.connect(s, t, WL.RULE_IDS[rule], weight=W, delay_ms=D, seed=23, **kw)
        b.finalize()
    rep = PU.compare_connections(g.read_connections(sorted=False), o.connections(sorted=False), 22.0, "node arrays, creation order")
    assert rep["n"] > 400_000 and rep["delay_mismatches"] == 0
    PU.compare_connections(g.read_connections(sorted=True), o.connections(sorted=True), 22.0, "node arrays, sorted")
    PU.compare_index(g.read_index(), o.index(), "node arrays")
    # bad ids are rejected with the oracle's code and leave the context usable
    g2, o2 = nc_mod.NC(), oracle_mod.Oracle()
    for b in (g2, o2):
        b.create_population(10)
        assert b.connect_rc(np.array([1, 10]), (0, 10), WL.RULE_IDS["all_to_all"]) == nc_mod.ERR_INVALID_ARG
        assert b.connect_rc(np.array([1, 2, 3]), np.array([4, 5]), WL.RULE_IDS["one_to_one"]) == nc_mod.ERR_INVALID_ARG
        assert b.num_connections() == 0
    g.close(); o.close(); g2.close(); o2.close()


def test_value_arrays_parity(nc_mod, oracle_mod):
    """nc_connect_values: per-connection weight and / or delay arrays, with ranges and with explicit
    node arrays, mixed with distribution projections, across several storage blocks -- bit-exact against the oracle
    (a given weight is stored as it is, a given delay goes through the fp64 rule D8), organised order and index too."""
    rng = np.random.default_rng(29)
    n_nodes = 2000
    ids = rng.choice(n_nodes, size=500, replace=False).astype(np.uint32)
    n1, n2, n3, n4 = 200_000, 500 * 31, 300, 64 * 90
    calls = [
        ((0, 2000), (0, 2000), "fixed_total_number", dict(degree_or_total=n1),
         dict(weights=rng.normal(0, 50, n1).astype(np.float32), delays=rng.uniform(0.0, 12.0, n1))),
        ((0, 2000), (0, 2000), "fixed_total_number", dict(degree_or_total=30_000), {}),
        ((100, 700), ids, "fixed_indegree", dict(degree_or_total=31), dict(weights=rng.normal(0, 1, n2).astype(np.float32))),
        (ids[:300], ids[200:500], "one_to_one", {}, dict(delays=rng.integers(1, 60, n3) * 0.1 + 0.05)),  # on boundaries
        (ids[:64], (0, 90), "all_to_all", {}, dict(weights=np.arange(n4, dtype=np.float32), delays=np.full(n4, 0.01))),
    ]
    o, g = oracle_mod.Oracle(dt_ms=0.1, block_size=50_000), nc_mod.NC(dt_ms=0.1, block_size=50_000)
    for b in (o, g):
        b.create_population(n_nodes)
        for s, t, rule, kw, vals in calls:
            b.connect(s, t, WL.RULE_IDS[rule], weight=W, delay_ms=D, seed=31, **kw, **vals)
        b.finalize()
    gu, ou = g.read_connections(sorted=False), o.connections(sorted=False)
    rep = PU.compare_connections(gu, ou, 22.0, "value arrays, creation order")
    assert rep["n"] == n1 + 30_000 + n2 + n3 + n4 and rep["delay_mismatches"] == 0
    # given values are exact, not merely within tolerance
    given = np.ones(rep["n"], dtype=bool)
    given[n1:n1 + 30_000] = False
    given[n1 + 30_000 + n2:n1 + 30_000 + n2 + n3] = False   # that projection gave delays only
    assert np.array_equal(gu["weight"][given], ou["weight"][given])
    PU.compare_connections(g.read_connections(sorted=True), o.connections(sorted=True), 22.0, "value arrays, sorted")
    PU.compare_index(g.read_index(), o.index(), "value arrays")
    # errors: same codes as the oracle, context left unchanged
    g2, o2 = nc_mod.NC(), oracle_mod.Oracle()
    ftn = WL.RULE_IDS["fixed_total_number"]
    for b in (g2, o2):
        b.create_population(20)
        assert b.connect_rc((0, 20), (0, 20), ftn, degree_or_total=10, weights=np.zeros(9)) == nc_mod.ERR_INVALID_ARG
        assert b.connect_rc((0, 20), (0, 20), ftn, degree_or_total=10, delays=np.full(10, np.nan)) == nc_mod.ERR_INVALID_ARG
        assert b.connect_rc((0, 20), (0, 20), ftn, degree_or_total=10, delays=np.full(10, 6553.6)) == nc_mod.ERR_CAPACITY
        assert b.connect_rc((0, 20), (0, 20), WL.RULE_IDS["pairwise_bernoulli"], p=0.5, weights=np.zeros(200)) == nc_mod.ERR_INVALID_ARG
        assert b.num_connections() == 0
    g.close(); o.close(); g2.close(); o2.close()


@pytest.mark.parametrize("variant", ["default", "pairs", "copass", "copass_shift"])
def test_connection_attributes_parity(nc_mod, oracle_mod, variant):
    """nc_set_connection_attributes / nc_read_connection_attributes (receptor port, synaptic group): the
    pair in force belongs to the connections of the following connect calls (an empty projection in between included)
    and is returned for the creation-order and the organised view, flat or inside the storage blocks."""
    flags = {"default": 0, "pairs": nc_mod.FLAG_SORT_PAIRS, "copass": nc_mod.FLAG_ORGANISE_COPASS,
             "copass_shift": nc_mod.FLAG_ORGANISE_COPASS | nc_mod.FLAG_COPASS_SHIFT}[variant]
    o, g = oracle_mod.Oracle(dt_ms=0.1, block_size=3000), nc_mod.NC(dt_ms=0.1, block_size=3000, flags=flags)
    calls = [((0, 0), "fixed_total_number", dict(degree_or_total=7000)), ((3, 0), "all_to_all", {}),
             ((9, 9), "pairwise_bernoulli", dict(p=0.0)),  # creates nothing
             ((255, 7), "pairwise_bernoulli", dict(p=0.3)), ((1, 1), "fixed_indegree", dict(degree_or_total=11))]
    for b in (o, g):
        b.create_population(120)
        for (port, group), rule, kw in calls:
            b.set_connection_attributes(port, group)
            b.connect((0, 120), (0, 120), WL.RULE_IDS[rule], weight=W, delay_ms=D, seed=5, **kw)
    po, go = o.read_connection_attributes(sorted=False)
    pg, gg = g.read_connection_attributes(sorted=False)
    assert np.array_equal(pg, po) and np.array_equal(gg, go) and set(po.tolist()) == {0, 3, 255, 1}
    for b in (o, g):
        b.finalize()
    PU.compare_connections(g.read_connections(sorted=True), o.connections(sorted=True), 22.0, "attributes " + variant)
    po, go = o.read_connection_attributes(sorted=True)
    pg, gg = g.read_connection_attributes(sorted=True)
    assert np.array_equal(pg, po) and np.array_equal(gg, go)
    p2, g2 = g.read_connection_attributes(sorted=True, first=4321, count=5000)
    assert np.array_equal(p2, po[4321:9321]) and np.array_equal(g2, go[4321:9321])
    g.close(); o.close()


def test_scratch_of_earlier_connect_calls_is_released(nc_mod):
    """Scratch queued for release (Bernoulli masks and tile tables, uploaded node and value arrays) goes back at the next
    point the stream is known idle, so the bytes held do not grow with the number of projections beyond the connections
    themselves (the masks of configs[4] would otherwise stay allocated through nc_finalize)."""
    g = nc_mod.NC(block_size=1 << 16)
    a = g.create_population(3000)
    held = []
    for k in range(6):
        g.connect((a, 3000), (a, 3000), nc_mod.PAIRWISE_BERNOULLI, p=0.01, weight=(1.0, 0.1, 0.0, math.inf),
                  delay_ms=(1.0, 0.2, 0.1, math.inf), seed=5)
        st = g.stats()
        held.append(st["bytes_in_use"] - st["n_blocks"] * 14 * (1 << 16))
    # one call's scratch (9e6 trials: 1.1 MB mask + tables) may be pending, never several
    assert max(held[1:]) <= held[0] + (1 << 20), held
    g.close()


def test_single_read_index_variant_parity(nc_mod, oracle_mod, monkeypatch):
    """NC_INDEX_FUSED=1: heads counted, chained across tiles by look-back and written by one kernel (one read of the
    organised keys instead of two).  Several tiles, sources without connections, a ragged last tile."""
    monkeypatch.setenv("NC_INDEX_FUSED", "1")
    for net in (WL.config2_microcircuit(scale=0.06), WL.config1_rule("fixed_outdegree", scale=0.2), WL.config0_tiny()):
        rep, _ = PU.full_parity(net, oracle_mod, nc_mod)
        assert rep["n"] >= 1000
