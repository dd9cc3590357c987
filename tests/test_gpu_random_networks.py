"""Randomised parity: seeded random sequences of populations and projections -- every rule, ranges and explicit node
arrays, distribution and per-connection value forms, E- and I-like weight signs, odd block sizes -- built on the CUDA path
under every organisation variant (default, (key, position) pairs, single-sweep look-back, COPASS by hole filling, COPASS
with the shift of Fig. 6E) and compared with the oracle element by element: creation order, organised order,
permutation, index, degree histograms."""
import math

import numpy as np
import pytest

from paper_2306_09855_b200 import workloads as WL
from tests import parity_util as PU

pytestmark = pytest.mark.gpu
INF = math.inf


@pytest.fixture(scope="module")
def nc_mod():
    from paper_2306_09855_b200 import binding, build
    build.build()
    return binding


def random_recipe(seed):
    """-> (population sizes, list of connect kwargs).  Sizes keep the oracle in the sub-second range."""
    rng = np.random.default_rng(seed)
    pops = [int(rng.integers(1, 400)) for _ in range(int(rng.integers(1, 6)))]
    first = np.concatenate([[0], np.cumsum(pops)])
    n_nodes = int(first[-1])
    calls = []
    for _ in range(int(rng.integers(1, 9))):
        def side():
            if rng.random() < 0.3:  # explicit node array: unsorted, may repeat
                return rng.integers(0, n_nodes, size=int(rng.integers(1, 300))).astype(np.uint32)
            p = int(rng.integers(0, len(pops)))
            lo = int(rng.integers(0, pops[p]))
            return (int(first[p]) + lo, int(rng.integers(1, pops[p] - lo + 1)))
        src, tgt = side(), side()
        n_src = src[1] if isinstance(src, tuple) else src.size
        n_tgt = tgt[1] if isinstance(tgt, tuple) else tgt.size
        rule = str(rng.choice(["one_to_one", "all_to_all", "fixed_indegree", "fixed_outdegree", "fixed_total_number",
                               "pairwise_bernoulli"]))
        kw, n_new = {}, None
        if rule == "one_to_one":
            m = min(n_src, n_tgt)
            src = (src[0], m) if isinstance(src, tuple) else src[:m]
            tgt = (tgt[0], m) if isinstance(tgt, tuple) else tgt[:m]
            n_new = m
        elif rule == "all_to_all":
            n_new = n_src * n_tgt
        elif rule == "fixed_indegree":
            kw["degree_or_total"] = int(rng.integers(1, 40))
            n_new = n_tgt * kw["degree_or_total"]
        elif rule == "fixed_outdegree":
            kw["degree_or_total"] = int(rng.integers(1, 40))
            n_new = n_src * kw["degree_or_total"]
        elif rule == "fixed_total_number":
            kw["degree_or_total"] = int(rng.integers(1, 20000))
            n_new = kw["degree_or_total"]
        else:
            kw["p"] = float(rng.choice([0.0, 0.01, 0.2, 0.7, 1.0]))
        exc = rng.random() < 0.7
        mean = float(rng.uniform(1, 100)) * (1 if exc else -4)
        kw["weight"] = (mean, abs(mean) * float(rng.choice([0.0, 0.1])), 0.0 if exc else -INF, INF if exc else 0.0)
        dm = float(rng.uniform(0.3, 3.0))
        kw["delay_ms"] = (dm, dm * float(rng.choice([0.0, 0.5])), 0.1, INF)
        kw["seed"] = int(rng.integers(0, 2**63))
        if n_new is not None and rng.random() < 0.25:  # per-connection value arrays
            if rng.random() < 0.7:
                kw["weights"] = rng.normal(0, 30, n_new).astype(np.float32)
            if "weights" not in kw or rng.random() < 0.5:
                kw["delays"] = rng.uniform(0.0, 8.0, n_new)
        calls.append((src, tgt, WL.RULE_IDS[rule], kw))
    return pops, calls


def build(b, pops, calls):
    for n in pops:
        b.create_population(n)
    for src, tgt, rule, kw in calls:
        b.connect(src, tgt, rule, **kw)


VARIANTS = ["default", "pairs", "onesweep", "bulk", "buckets", "copass", "copass_shift"]


@pytest.mark.parametrize("seed", range(24))
def test_random_network_all_variants(nc_mod, oracle_mod, seed):
    pops, calls = random_recipe(1000 + seed)
    rng = np.random.default_rng(seed)
    B = int(rng.choice([0, 1 << 12, 1000, 4097, 257]))
    flags = {"default": 0, "pairs": nc_mod.FLAG_SORT_PAIRS, "onesweep": nc_mod.FLAG_SORT_ONESWEEP, "bulk": nc_mod.FLAG_SORT_BULK,
             "buckets": nc_mod.FLAG_SORT_BUCKETS, "copass": nc_mod.FLAG_ORGANISE_COPASS, "copass_shift": nc_mod.FLAG_ORGANISE_COPASS | nc_mod.FLAG_COPASS_SHIFT}
    o = oracle_mod.Oracle(dt_ms=0.1, block_size=B)
    build(o, pops, calls)
    ou = o.connections(sorted=False)
    n = ou["n"]
    o.finalize()
    os_, oi = o.connections(sorted=True), o.index()
    per_proj = [abs(kw["weight"][0]) + kw["weight"][1] for _, _, _, kw in calls]  # the synapse's own projection scale
    scale = PU.scale_per_connection(per_proj, o)
    scale_s = scale[os_["perm"]]
    for name in VARIANTS:
        if name.startswith("copass") and B and (n + B - 1) // B > 4096:
            continue
        g = nc_mod.NC(dt_ms=0.1, block_size=B, flags=flags[name])
        build(g, pops, calls)
        assert g.num_connections() == n, name
        if n:
            rep = PU.compare_connections(g.read_connections(sorted=False), ou, scale, f"seed {seed} {name} creation order")
            ind = g.read_degree_histogram(0)
            od, om = o.degree_histogram(0)
            assert np.array_equal(ind[0], od) and ind[1] == om, name
        g.finalize()
        assert g.stats()["n_blocks"] == o.num_blocks(), name
        if n and rep["delay_mismatches"] == 0:
            PU.compare_connections(g.read_connections(sorted=True), os_, scale_s, f"seed {seed} {name} organised")
        PU.compare_index(g.read_index(), oi, f"seed {seed} {name}") if (n == 0 or rep["delay_mismatches"] == 0) else None
        outd = g.read_degree_histogram(1)
        od, om = o.degree_histogram(1)
        assert np.array_equal(outd[0], od) and outd[1] == om, name
        g.close()
    o.close()
