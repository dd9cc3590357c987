"""Seeded synthetic workload recipes (BASELINE.json configs 0-4) -- input generators only.

This module holds NONE of the method's arithmetic (no RNG, no rule expansion, no transforms, no
sort): it only lists populations and connect calls.  It serves both the CUDA path and the test
oracle, which is why it imports neither.  `run(net, backend)` replays a recipe on any object with
`create_population(n)`, `connect(src, tgt, rule, ...)` and `finalize()` -- the nc_ binding and
the oracle binding both have that shape.

The recipes stand in for the paper's workloads (PAPER.md:140 cortical microcircuit built with
fixed_total_number; PAPER.md:148-162 two-population scaling network); nothing external is read.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field
from typing import List, Tuple

INF = math.inf

RULE_IDS = {
    "one_to_one": 0,
    "all_to_all": 1,
    "fixed_indegree": 2,
    "fixed_outdegree": 3,
    "fixed_total_number": 4,
    "pairwise_bernoulli": 5,
}

Dist = Tuple[float, float, float, float]  # (mean, sd, lo, hi): normal clamped to [lo, hi]


@dataclass
class Projection:
    src_pop: int
    tgt_pop: int
    rule: str
    degree_or_total: int = 0
    p: float = 0.0
    weight: Dist = (1.0, 0.0, -INF, INF)
    delay_ms: Dist = (1.0, 0.0, -INF, INF)
    seed: int = 0


@dataclass
class Network:
    name: str
    populations: List[int]
    projections: List[Projection] = field(default_factory=list)
    dt_ms: float = 0.1

    @property
    def n_nodes(self) -> int:
        return sum(self.populations)

    def expected_connections(self):
        """Exact synapse count when no projection is pairwise_bernoulli, else the binomial mean."""
        tot = 0.0
        for pr in self.projections:
            ns, nt = self.populations[pr.src_pop], self.populations[pr.tgt_pop]
            tot += {
                "one_to_one": ns,
                "all_to_all": ns * nt,
                "fixed_indegree": nt * pr.degree_or_total,
                "fixed_outdegree": ns * pr.degree_or_total,
                "fixed_total_number": pr.degree_or_total,
                "pairwise_bernoulli": ns * nt * pr.p,
            }[pr.rule]
        return tot


def signed_weight(mean: float, rel_sd: float = 0.1) -> Dist:
    """'sign-clipped' normal (BASELINE.json): lo = 0 for positive mean, hi = 0 for negative mean (Q19)."""
    sd = abs(mean) * rel_sd
    if mean > 0:
        return (mean, sd, 0.0, INF)
    if mean < 0:
        return (mean, sd, -INF, 0.0)
    return (mean, sd, -INF, INF)


def delay(mean: float, sd: float, lo: float = 0.1) -> Dist:
    return (mean, sd, lo, INF)


def run(net: Network, backend, finalize: bool = True, shard=None):
    """Replay the recipe: populations in listed order, projections in listed order (projection_id =
    issue order).  shard = (first node id, count): the backend keeps only the connections whose target
    it owns (nc_set_shard)."""
    firsts = [backend.create_population(n) for n in net.populations]
    if shard is not None:
        backend.set_shard(*shard)
    for pr in net.projections:
        backend.connect(
            (firsts[pr.src_pop], net.populations[pr.src_pop]),
            (firsts[pr.tgt_pop], net.populations[pr.tgt_pop]),
            RULE_IDS[pr.rule],
            degree_or_total=pr.degree_or_total,
            p=pr.p,
            weight=pr.weight,
            delay_ms=pr.delay_ms,
            seed=pr.seed,
        )
    if finalize:
        backend.finalize()
    return firsts


# ------------------------------------------------------------------------------------------
# two-population networks (configs 0, 1, 3, 4)
# ------------------------------------------------------------------------------------------

def _two_pop(name, n_e, n_i, rule, seed, k_e=0, k_i=0, total=0, p=0.0, w_e=20.0, w_i=-80.0,
             pairs=((0, 0), (0, 1), (1, 0), (1, 1))):
    """E->E, E->I, I->E, I->I (issue order of SURVEY.md 8(d)); K/N depends on the SOURCE population."""
    net = Network(name, [n_e, n_i])
    for s, t in pairs:
        k = (k_e, k_i)[s]
        net.projections.append(Projection(
            s, t, rule,
            degree_or_total=total if rule == "fixed_total_number" else k,
            p=p,
            weight=signed_weight((w_e, w_i)[s]),
            delay_ms=delay(1.5, 0.75),
            seed=seed))
    return net


def config0_tiny() -> Network:
    """configs[0]: E=80, I=20, fixed_indegree K_E=8 / K_I=2, seed 1234 -> 1,000 synapses."""
    return _two_pop("c0_tiny", 80, 20, "fixed_indegree", 1234, k_e=8, k_i=2)


def config1_rule(rule: str, n_e: int = 8000, n_i: int = 2000, scale: float = 1.0) -> Network:
    """configs[1]: one run per rule, E=8,000, I=2,000, seed 42.  `scale` < 1 shrinks populations and
    degrees together (test sizes); scale = 1 is the config as written."""
    n_e = max(1, int(round(n_e * scale)))
    n_i = max(1, int(round(n_i * scale)))
    sc = lambda v: max(1, int(round(v * scale)))  # noqa: E731
    name = f"c1_{rule}" + ("" if scale == 1.0 else f"_x{scale:g}")
    if rule == "one_to_one":
        return _two_pop(name, n_e, n_i, rule, 42, pairs=((0, 0),))
    if rule == "all_to_all":
        return _two_pop(name, n_e, n_i, rule, 42)
    if rule == "fixed_indegree":
        return _two_pop(name, n_e, n_i, rule, 42, k_e=sc(800), k_i=sc(200))
    if rule == "fixed_outdegree":
        return _two_pop(name, n_e, n_i, rule, 42, k_e=sc(1000), k_i=sc(1000))
    if rule == "fixed_total_number":
        return _two_pop(name, n_e, n_i, rule, 42, total=max(1, int(round(10_000_000 * scale * scale))))
    if rule == "pairwise_bernoulli":
        return _two_pop(name, n_e, n_i, rule, 42, p=0.1)
    raise ValueError(rule)


def config3_large_indegree(scale: float = 1.0) -> Network:
    """configs[3]: E=80,000, I=20,000, fixed_indegree K=8,000 from E / 2,000 from I, seed 99 -> 1e9."""
    sc = lambda v: max(1, int(round(v * scale)))  # noqa: E731
    return _two_pop("c3_large_indegree" + ("" if scale == 1.0 else f"_x{scale:g}"), sc(80_000), sc(20_000),
                    "fixed_indegree", 99, k_e=sc(8000), k_i=sc(2000))


def config4_large_bernoulli(scale: float = 1.0) -> Network:
    """configs[4]: E=160,000, I=40,000, 4x pairwise_bernoulli p=0.025 + fixed_outdegree E->E K=500, seed 2023."""
    sc = lambda v: max(1, int(round(v * scale)))  # noqa: E731
    net = _two_pop("c4_large_bernoulli" + ("" if scale == 1.0 else f"_x{scale:g}"), sc(160_000), sc(40_000),
                   "pairwise_bernoulli", 2023, p=0.025)
    net.projections.append(Projection(0, 0, "fixed_outdegree", degree_or_total=sc(500),
                                      weight=signed_weight(20.0), delay_ms=delay(1.5, 0.75), seed=2023))
    return net


# ------------------------------------------------------------------------------------------
# cortical-microcircuit-shaped network (config 2)
# ------------------------------------------------------------------------------------------

MICROCIRCUIT_POPS = ("L2/3E", "L2/3I", "L4E", "L4I", "L5E", "L5I", "L6E", "L6I")
MICROCIRCUIT_SIZES = (20683, 5834, 21915, 5479, 4850, 1065, 14395, 2948)
# connection probabilities, rows = targets, columns = sources (BASELINE.json configs[2])
MICROCIRCUIT_P = (
    (.1009, .1689, .0437, .0818, .0323, 0., .0076, 0.),
    (.1346, .1371, .0316, .0515, .0755, 0., .0042, 0.),
    (.0077, .0059, .0497, .1350, .0067, .0003, .0453, 0.),
    (.0691, .0029, .0794, .1597, .0033, 0., .1057, 0.),
    (.1004, .0622, .0505, .0057, .0831, .3726, .0204, 0.),
    (.0548, .0269, .0257, .0022, .0600, .3158, .0086, 0.),
    (.0156, .0066, .0211, .0166, .0572, .0197, .0396, .2252),
    (.0364, .0010, .0034, .0005, .0277, .0080, .0658, .1443),
)


def fixed_total_from_probability(p: float, n_pre: int, n_post: int) -> int:
    """N = round(log(1-p) / log(1 - 1/(Npre*Npost))) (BASELINE.json configs[2]), evaluated with log1p in
    fp64 and rounded half away from zero (reading Q16).  Computed ONCE here and handed as the same
    integer to the CUDA path and to the oracle."""
    if p <= 0.0:
        return 0
    x = math.log1p(-p) / math.log1p(-1.0 / (float(n_pre) * float(n_post)))
    return int(math.floor(x + 0.5))


def config2_microcircuit(scale: float = 1.0) -> Network:
    """configs[2]: 8 populations, 55 non-zero (target, source) pairs issued row-major (target row,
    source column), fixed_total_number, seed 7.  scale = 1 -> 77,169 nodes, 298,880,970 synapses."""
    sizes = [max(1, int(round(n * scale))) for n in MICROCIRCUIT_SIZES]
    net = Network("c2_microcircuit" + ("" if scale == 1.0 else f"_x{scale:g}"), sizes)
    for t in range(8):
        for s in range(8):
            p = MICROCIRCUIT_P[t][s]
            n = fixed_total_from_probability(p, sizes[s], sizes[t])
            if n == 0:
                continue
            excit = (s % 2 == 0)
            w_mean = 87.8 if excit else -351.2
            if s == 2 and t == 0:  # L4E -> L2/3E doubled (BASELINE.json configs[2])
                w_mean *= 2.0
            d = delay(1.5, 0.75) if excit else delay(0.75, 0.375)
            net.projections.append(Projection(s, t, "fixed_total_number", degree_or_total=n,
                                              weight=signed_weight(w_mean), delay_ms=d, seed=7))
    return net


def by_name(name: str, **kw) -> Network:
    if name == "c0":
        return config0_tiny()
    if name.startswith("c1:"):
        return config1_rule(name[3:], **kw)
    if name == "c2":
        return config2_microcircuit(**kw)
    if name == "c3":
        return config3_large_indegree(**kw)
    if name == "c4":
        return config4_large_bernoulli(**kw)
    raise ValueError(name)
