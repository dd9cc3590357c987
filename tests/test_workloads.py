"""The synthetic workload recipes reproduce the sizes BASELINE.json / the paper state.  CPU only."""
import math

from paper_2306_09855_b200 import workloads as WL


def test_microcircuit_totals():
    """'about 77,000 neurons ... 300 million synapses'; 77,169 nodes, 55
    non-zero projections, 298,880,970 synapses with log1p evaluation, min 7,003, max 45,499,806."""
    net = WL.config2_microcircuit()
    ns = [p.degree_or_total for p in net.projections]
    assert net.n_nodes == 77169 and len(ns) == 55
    assert sum(ns) == 298_880_970 and min(ns) == 7003 and max(ns) == 45_499_806
    # issue order: row-major over (target row, source column); first is L2/3E -> L2/3E
    assert (net.projections[0].src_pop, net.projections[0].tgt_pop) == (0, 0)
    assert (net.projections[1].src_pop, net.projections[1].tgt_pop) == (1, 0)
    dbl = [p for p in net.projections if p.src_pop == 2 and p.tgt_pop == 0][0]
    assert dbl.weight[0] == 175.6 and abs(dbl.weight[1] - 17.56) < 1e-12
    inh = [p for p in net.projections if p.src_pop == 1][0]
    assert inh.weight == (-351.2, 35.120000000000005, -math.inf, 0.0) or abs(inh.weight[1] - 35.12) < 1e-9
    assert inh.delay_ms[:3] == (0.75, 0.375, 0.1)
    # the naive log(1-x) form loses digits (Q16): log1p is what the recipe uses
    assert WL.fixed_total_from_probability(0.1009, 20683, 20683) == 45_499_806


def test_two_population_sizes():
    assert WL.config0_tiny().expected_connections() == 1000
    assert WL.config1_rule("one_to_one").expected_connections() == 8000
    assert WL.config1_rule("all_to_all").expected_connections() == 10**8
    assert WL.config1_rule("fixed_indegree").expected_connections() == 10**7
    assert WL.config1_rule("fixed_outdegree").expected_connections() == 2 * 10**7
    assert WL.config1_rule("fixed_total_number").expected_connections() == 4 * 10**7
    assert abs(WL.config1_rule("pairwise_bernoulli").expected_connections() - 10**7) < 1
    assert WL.config3_large_indegree().expected_connections() == 10**9
    c4 = WL.config4_large_bernoulli()
    assert abs(c4.expected_connections() - (4e10 * 0.025 + 8e7)) < 1 and len(c4.projections) == 5
    assert [(p.src_pop, p.tgt_pop) for p in WL.config0_tiny().projections] == [(0, 0), (0, 1), (1, 0), (1, 1)]
