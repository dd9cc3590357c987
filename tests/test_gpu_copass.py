"""GPU parity of the COPASS block-sort (include/nc_copass.h): the partition kernel against the
oracle's step-by-step partition (oracle/copass.cpp) on inputs with long runs of ties, empty subarrays and many
subarrays; the in-place organisation (NC_FLAG_ORGANISE_COPASS) against the oracle's organised connections and index,
element by element."""
from pathlib import Path

import numpy as np
import pytest

from paper_2306_09855_b200 import workloads as WL
from tests import parity_util as PU

pytestmark = pytest.mark.gpu
GOLDEN = Path(__file__).parent / "golden" / "copass_partition.txt"


@pytest.fixture(scope="module")
def nc_mod():
    from paper_2306_09855_b200 import binding, build
    build.build()
    return binding


def _flatten(subs):
    lens = np.array([len(s) for s in subs], dtype=np.uint32)
    start = np.concatenate([[0], np.cumsum(lens)[:-1]]).astype(np.uint32)
    keys = np.concatenate([np.asarray(s, dtype=np.uint32) for s in subs])
    return keys, start, lens


def _both(g, oracle_mod, subs, m):
    keys, start, lens = _flatten(subs)
    got = g.copass_partition(keys, start, lens, m)
    want = oracle_mod.copass_partition(keys.astype(np.int64), start, lens, m)
    assert got[0].tolist() == want[0].astype(int).tolist(), (m, got, want)
    assert got[1:] == want[1:], (m, got, want)  # threshold, iteration count, which last step
    return got


def test_partition_golden_cases_on_device(nc_mod, oracle_mod):
    g = nc_mod.NC()
    for line in [l for l in GOLDEN.read_text().splitlines() if l and not l.startswith("#")]:
        name, subs, m, want, t, it, last = [f.strip() for f in line.split("|")]
        subs = [[int(x) for x in s.split()] for s in subs.split(";")]
        keys, start, lens = _flatten(subs)
        m_i, got_t, got_it, got_last = g.copass_partition(keys, start, lens, int(m))
        assert m_i.tolist() == [int(x) for x in want.split()], name
        assert (got_t, got_it, got_last) == (int(t), int(it), int(last)), name
    g.close()


@pytest.mark.parametrize("seed", range(8))
def test_partition_matches_oracle_small_with_ties(nc_mod, oracle_mod, seed):
    rng = np.random.default_rng(seed)
    g = nc_mod.NC()
    seen = set()
    for _ in range(12):
        k = int(rng.integers(1, 12))
        span = int(rng.choice([2, 6, 60, 2**32 - 1]))
        subs = [np.sort(rng.integers(0, span, size=int(rng.integers(0, 70)))) for _ in range(k)]
        total = sum(len(s) for s in subs)
        if total < 2:
            continue
        for m in sorted(set([1, total - 1] + rng.integers(1, total, size=4).tolist())):
            seen.add(_both(g, oracle_mod, subs, m)[3])
    assert seen == {1, 2}
    g.close()


def test_partition_matches_oracle_large(nc_mod, oracle_mod):
    """Sizes at which every search takes several 32-ary steps; many subarrays (more than the CTA has warps, and
    more than it has threads); keys at both ends of the 32-bit range."""
    rng = np.random.default_rng(42)
    g = nc_mod.NC()
    # 40 subarrays of ~50,000 keys: (source << 6 | delay)-like keys with runs of equal keys
    subs = [np.sort(rng.integers(0, 2**16, size=int(rng.integers(30000, 70000)))) for _ in range(40)]
    total = sum(len(s) for s in subs)
    for m in (1, 77, total // 3, total // 2 + 1, total - 1):
        _both(g, oracle_mod, subs, m)
    # 1500 and 4096 short subarrays, some of them empty
    for k in (1500, 4096):
        subs = [np.sort(rng.integers(0, 2**32 - 1, size=int(rng.integers(0, 40)))) for _ in range(k)]
        subs[0] = np.array([0, 0, 2**32 - 1], dtype=np.uint64)
        total = sum(len(s) for s in subs)
        for m in (1, total // 2, total - 1):
            _both(g, oracle_mod, subs, m)
    # all keys equal: Sec. A4 in the first iteration, the d_i handed out lowest subarray first
    subs = [np.full(1000, 7)] * 5
    got = _both(g, oracle_mod, subs, 2500)
    assert got[0].tolist() == [1000, 1000, 500, 0, 0] and got[3] == 2
    g.close()


def test_partition_argument_errors(nc_mod):
    g = nc_mod.NC()
    keys, start, lens = _flatten([[1, 2, 3], [4, 5]])
    for m in (0, 5, 9):
        with pytest.raises(nc_mod.NCError) as e:
            g.copass_partition(keys, start, lens, m)
        assert e.value.code == nc_mod.ERR_INVALID_ARG
    with pytest.raises(nc_mod.NCError) as e:
        g.copass_partition(keys, [0, 3], [3, 5], 2)  # second subarray runs past the keys
    assert e.value.code == nc_mod.ERR_INVALID_ARG
    g.close()


def copass_parity(net, oracle_mod, nc_mod, B, shift=False):
    o = oracle_mod.Oracle(dt_ms=net.dt_ms, block_size=B)
    WL.run(net, o, finalize=True)
    flags = nc_mod.FLAG_ORGANISE_COPASS | (nc_mod.FLAG_COPASS_SHIFT if shift else 0)
    g = nc_mod.NC(dt_ms=net.dt_ms, block_size=B, flags=flags)
    WL.run(net, g, finalize=False)
    gu = g.read_connections(sorted=False)
    rep = PU.compare_connections(gu, o.connections(sorted=False), PU.weight_scale(net, o), net.name + " creation order")
    in_deg = g.read_degree_histogram(0)
    g.finalize()
    gs = g.read_connections(sorted=True)
    if rep["delay_mismatches"] == 0:
        os_ = o.connections(sorted=True)
        PU.compare_connections(gs, os_, PU.weight_scale(net, o, os_["perm"]), net.name + " organised in place")
        PU.compare_index(g.read_index(), o.index(), net.name)
    else:  # a boundary delay moved by one step: the order is the stable sort of the device's own keys
        key = (gu["source"].astype(np.uint64) << np.uint64(16)) | gu["delay"].astype(np.uint64)
        perm = np.argsort(key, kind="stable").astype(np.uint32)
        assert np.array_equal(gs["perm"], perm)
        for f in ("source", "target", "weight", "delay"):
            assert np.array_equal(gs[f], gu[f][perm]), f
    # the blocks were sorted in place: the creation-order view is gone, the block structure is kept
    with pytest.raises(nc_mod.NCError) as e:
        g.read_connections(sorted=False)
    assert e.value.code == nc_mod.ERR_STATE
    st = g.copass_stats()
    n = rep["n"]
    block = B if B else 1 << 24
    k = (n + block - 1) // block
    assert st["n_blocks"] == k == o.num_blocks()
    assert st["partitions"] == max(k - 1, 0) == st["last_step_1"] + st["last_step_2"]
    v = g.get_connections(sorted=True)
    assert v.n_blocks == k and v.block_size == block and v.off_perm > v.off_delay
    # degree histograms still count over the blocks
    od, om = o.degree_histogram(0)
    assert np.array_equal(in_deg[0], od) and in_deg[1] == om
    gd, gm = g.read_degree_histogram(0)
    assert np.array_equal(gd, od) and gm == om
    gd, gm = g.read_degree_histogram(1)
    od, om = o.degree_histogram(1)
    assert np.array_equal(gd, od) and gm == om
    g.close()
    return rep, st


@pytest.mark.parametrize("shift", [False, True], ids=["fill", "shift"])
@pytest.mark.parametrize("B", [0, 1, 7, 10, 64, 250, 999, 1000])
def test_copass_config0_tiny(nc_mod, oracle_mod, B, shift):
    """shift = Fig. 6 C-E to the letter; fill = the default extraction by hole filling"""
    rep, st = copass_parity(WL.config0_tiny(), oracle_mod, nc_mod, B, shift)
    assert rep["n"] == 1000


@pytest.mark.parametrize("rule,scale,B", [("one_to_one", 1.0, 1000), ("all_to_all", 0.15, 300_000),
                                          ("fixed_indegree", 0.3, 100_000), ("fixed_outdegree", 0.25, 131_072),
                                          ("fixed_total_number", 0.3, 250_001), ("pairwise_bernoulli", 0.4, 65_536)])
@pytest.mark.parametrize("shift", [False, True], ids=["fill", "shift"])
def test_copass_config1_rules(nc_mod, oracle_mod, rule, scale, B, shift):
    """Several sort tiles per block, a ragged last block, block sizes that are and are not powers of two."""
    net = WL.config1_rule(rule, scale=scale)
    rep, st = copass_parity(net, oracle_mod, nc_mod, B, shift)
    print(net.name, rep, st)
    assert st["n_blocks"] >= 3


def test_copass_microcircuit_scaled(nc_mod, oracle_mod):
    """configs[2] at 10 % of the populations, ~3e6 connections in 12 blocks of 2^18."""
    net = WL.config2_microcircuit(scale=0.1)
    for shift in (False, True):
        rep, st = copass_parity(net, oracle_mod, nc_mod, 1 << 18, shift)
        print(rep, st)
    assert st["n_blocks"] >= 10 and st["iterations"] >= st["partitions"]


def test_copass_uses_a_few_blocks_of_auxiliary_memory(nc_mod):
    """The point of the algorithm: the organisation step holds a few blocks, not copies of all
    connections.  2e6 connections in blocks of 2^16: the default path's scratch is > 50 B per connection."""
    net = WL.config1_rule("fixed_total_number", scale=0.2)
    B = 1 << 16
    g = nc_mod.NC(dt_ms=net.dt_ms, block_size=B, flags=nc_mod.FLAG_ORGANISE_COPASS)
    WL.run(net, g, finalize=True)
    st = g.copass_stats()
    n = g.num_connections()
    assert st["n_blocks"] == (n + B - 1) // B >= 20
    assert st["aux_bytes"] <= 80 * B + (1 << 20)   # 18 (spare) + 16 (aux) + 33 (sort scratch) B per entry of ONE block
    assert st["aux_bytes"] < 0.1 * 50 * n
    g.close()


def test_delivery_over_copass_blocks(nc_mod, oracle_mod):
    """Spike delivery (include/nc_delivery.h) over connections organised inside 10 storage blocks: groups straddle
    blocks; the spike array and every node's input equal the oracle's step by step."""
    import torch
    net = WL.config0_tiny()
    o = oracle_mod.Oracle(dt_ms=net.dt_ms, block_size=100)
    WL.run(net, o)
    g = nc_mod.NC(dt_ms=net.dt_ms, block_size=100, flags=nc_mod.FLAG_ORGANISE_COPASS)
    WL.run(net, g)
    od, gd = oracle_mod.Delivery(o), nc_mod.Delivery(g, 4096)
    inp = torch.zeros(net.n_nodes, dtype=torch.float32, device="cuda")
    rng = np.random.default_rng(4)
    for k in range(80):
        nodes = rng.choice(net.n_nodes, size=int(rng.integers(0, 12)) if k < 30 else 0, replace=False).astype(np.uint32)
        want = np.zeros(net.n_nodes)
        od.step(nodes, None, want)
        inp.zero_()
        gd.step(torch.from_numpy(nodes.astype(np.int32)).cuda(), None, inp)
        go, gm = gd.read_spike_array()
        wo, wm = od.spike_array()
        assert sorted(zip(go.tolist(), gm.tolist())) == sorted(zip(wo.tolist(), wm.tolist())), k
        assert np.abs(inp.cpu().numpy() - want).max() <= 1e-5 * max(1.0, np.abs(want).max()), k
    assert gd.counts()["events"] == od.counts()[1] > 0
    gd.close(); od.close(); g.close(); o.close()


def test_copass_full_size_microcircuit(nc_mod):
    """configs[2] at FULL size (298,880,970 connections, 18 blocks of 2^24) organised in place, in the configuration
    `bench.py --flags 16` times.  The oracle cannot hold this network in seconds, so the organised blocks are checked
    against the plain definitions (readings D10, D11) evaluated with numpy on the device's own creation-order arrays,
    read before nc_finalize: permutation, order, stability, every gathered field, every index array."""
    net = WL.config2_microcircuit()
    g = nc_mod.NC(dt_ms=net.dt_ms, flags=nc_mod.FLAG_ORGANISE_COPASS)
    WL.run(net, g, finalize=False)
    n = g.num_connections()
    assert n == 298_880_970
    u = g.read_connections(sorted=False)
    g.finalize()
    st = g.copass_stats()
    print(st, g.stats())
    assert st["n_blocks"] == 18 and st["partitions"] == 17
    assert st["aux_bytes"] < 80 * (1 << 24) + (1 << 22)
    assert g.stats()["bytes_peak"] < 18 * n + st["aux_bytes"] + (1 << 28)   # never a second copy of the connections
    s = g.read_connections(sorted=True)
    perm = s["perm"]
    seen = np.zeros(n, dtype=bool)
    seen[perm] = True
    assert seen.all(), "perm is not a permutation"
    del seen
    key = (s["source"].astype(np.uint64) << np.uint64(16)) | s["delay"].astype(np.uint64)
    dk = key[1:] != key[:-1]
    assert np.all(key[1:] >= key[:-1]), "not sorted by (source, delay)"
    assert np.all(dk | (perm[1:] > perm[:-1])), "ties are not in creation order"
    del key
    for f in ("source", "target", "weight", "delay"):
        assert np.array_equal(u[f][perm], s[f]), f
    idx = g.read_index()
    out_deg = np.bincount(s["source"], minlength=net.n_nodes)
    assert np.array_equal(idx["src_offsets"], np.concatenate([[0], np.cumsum(out_deg)]).astype(np.uint32))
    heads = np.concatenate([[0], np.flatnonzero(dk) + 1]).astype(np.uint32)
    assert idx["total_groups"] == heads.size
    assert np.array_equal(idx["group_start"], heads)
    assert np.array_equal(idx["group_delay"], s["delay"][heads])
    gcount = np.bincount(s["source"][heads], minlength=net.n_nodes).astype(np.uint32)
    assert np.array_equal(idx["group_count"], gcount)
    assert np.array_equal(idx["group_ptr"], np.concatenate([[0], np.cumsum(gcount)]).astype(np.uint32))
    g.close()


def test_copass_capacity_errors_leave_the_connections_intact(nc_mod, oracle_mod):
    """More than 4096 blocks: NC_ERR_CAPACITY before anything is rewritten -- the creation-order view still reads."""
    g = nc_mod.NC(dt_ms=0.1, block_size=1, flags=nc_mod.FLAG_ORGANISE_COPASS)
    o = oracle_mod.Oracle(dt_ms=0.1, block_size=1)
    for b in (g, o):
        b.create_population(50)
        b.connect((0, 50), (0, 50), WL.RULE_IDS["fixed_total_number"], degree_or_total=5000, weight=(1.0, 0.1, 0.0, float("inf")),
                  delay_ms=(1.5, 0.75, 0.1, float("inf")), seed=8)
    with pytest.raises(nc_mod.NCError) as e:
        g.finalize()
    assert e.value.code == nc_mod.ERR_CAPACITY
    PU.compare_connections(g.read_connections(sorted=False), o.connections(sorted=False), 1.1, "after a refused finalize")
    g.close(); o.close()


@pytest.mark.parametrize("shift", [False, True], ids=["fill", "shift"])
def test_copass_single_digit_pass_key(nc_mod, oracle_mod, shift):
    """Four nodes and delays of at most 7 steps: the (source, delay) key has 5 bits, the underlying sort is ONE digit
    pass -- the path where a sorted block cannot be written over its own input."""
    flags = nc_mod.FLAG_ORGANISE_COPASS | (nc_mod.FLAG_COPASS_SHIFT if shift else 0)
    o, g = oracle_mod.Oracle(dt_ms=0.1, block_size=300), nc_mod.NC(dt_ms=0.1, block_size=300, flags=flags)
    for b in (o, g):
        b.create_population(4)
        b.connect((0, 4), (0, 4), WL.RULE_IDS["fixed_total_number"], degree_or_total=2500, weight=(1.0, 0.2, 0.0, float("inf")),
                  delay_ms=(0.4, 0.1, 0.1, 0.7), seed=12)
        b.finalize()
    st = g.stats()
    assert st["sort_passes"] == 1 and st["key_bits"] <= 8
    PU.compare_connections(g.read_connections(sorted=True), o.connections(sorted=True), 2.0, "single pass")
    PU.compare_index(g.read_index(), o.index(), "single pass")
    assert g.copass_stats()["n_blocks"] == 9
    g.close(); o.close()


@pytest.mark.parametrize("shift", [False, True], ids=["fill", "shift"])
def test_copass_with_the_library_allocator(nc_mod, oracle_mod, shift):
    """mem.alloc == NULL: cudaMalloc / cudaFree inside the library (no caching allocator underneath the block swaps)."""
    net = WL.config1_rule("fixed_outdegree", scale=0.1)
    o = oracle_mod.Oracle(dt_ms=net.dt_ms, block_size=40_000)
    WL.run(net, o)
    flags = nc_mod.FLAG_ORGANISE_COPASS | (nc_mod.FLAG_COPASS_SHIFT if shift else 0)
    g = nc_mod.NC(dt_ms=net.dt_ms, block_size=40_000, flags=flags, use_torch_allocator=False)
    WL.run(net, g)
    PU.compare_sorted(g, o, net, "cudaMalloc")
    PU.compare_index(g.read_index(), o.index(), "cudaMalloc")
    assert g.copass_stats()["n_blocks"] >= 4
    g.close(); o.close()
