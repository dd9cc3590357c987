"""Pins of the oracle's autapse / multapse prohibition (readings A1-A6 in oracle/oracle.h): what the flags
mean is fixed by things other than the oracle's own arithmetic -- no pair with equal ids, no repeated pair, exact degrees
kept, the unflagged result wherever it was already allowed, set identities against the unflagged rules, a brute-force
bijection check of the keyed permutation, chi-square uniformity over the allowed partners."""
import math

import numpy as np
import pytest

import oracle as O

W = (1.0, 0.1, 0.0, math.inf)
D = (1.5, 0.75, 0.1, math.inf)
R = dict(one_to_one=0, all_to_all=1, fixed_indegree=2, fixed_outdegree=3, fixed_total_number=4, pairwise_bernoulli=5)


def build(n_nodes, src, tgt, rule, flags, seed=11, **kw):
    o = O.Oracle(dt_ms=0.1)
    o.create_population(n_nodes)
    o.set_rule_flags(flags)
    o.connect(src, tgt, R[rule], weight=W, delay_ms=D, seed=seed, **kw)
    c = o.connections(sorted=False)
    out = {k: np.array(c[k]) for k in ("source", "target", "weight", "delay")}
    o.close()
    return out


def chi2_ok(counts, expected, sigmas=5.0):
    counts = np.asarray(counts, dtype=np.float64)
    chi2 = float(((counts - expected) ** 2 / expected).sum())
    dof = counts.size - 1
    return abs(chi2 - dof) <= sigmas * math.sqrt(2 * dof) + 1e-9


def test_keyed_permutation_is_a_bijection_brute_force():
    rng = np.random.default_rng(3)
    for M in list(range(1, 70)) + [127, 128, 129, 255, 256, 257, 1000, 4097, 65535, 65536, 65537]:
        keys = rng.integers(0, 2**32, size=4, dtype=np.uint64)
        img = sorted(O.keyed_permutation(M, k, keys) for k in range(M))
        assert img == list(range(M)), M


def test_keyed_permutation_hand_iterated_case():
    """M = 6 -> bits(5) = 3, h = 2, mask = 3, domain 16.  The Feistel rounds and the cycle walk re-done here in Python
    from the definition in oracle.h."""
    def mix32(v):
        v &= 0xffffffff
        v ^= v >> 16
        v = (v * 0x7feb352d) & 0xffffffff
        v ^= v >> 15
        v = (v * 0x846ca68b) & 0xffffffff
        v ^= v >> 16
        return v
    keys = [0x12345678, 0x9abcdef0, 0x0f1e2d3c, 0xdeadbeef]
    for M, h in ((6, 2), (2, 1), (17, 3), (300, 5), (70000, 9)):
        mask = (1 << h) - 1
        for k in range(min(M, 40)):
            x = k
            while True:
                L, Rr = x >> h, x & mask
                for r in range(6 + -(-24 // h)):
                    key_r = (keys[r & 3] + r * 0x9E3779B9) & 0xffffffff
                    L, Rr = Rr, L ^ (mix32(Rr ^ key_r) & mask)
                x = (L << h) | Rr
                if x < M:
                    break
            assert O.keyed_permutation(M, k, keys) == x, (M, k)


@pytest.mark.parametrize("rule,kw", [("all_to_all", {}), ("one_to_one", {}), ("pairwise_bernoulli", dict(p=0.3)),
                                     ("pairwise_bernoulli", dict(p=1.0))])
def test_a2_rules_drop_exactly_the_equal_id_pairs(rule, kw):
    """A2: the flagged call equals the unflagged call with the autapses removed, order, weights and delays included."""
    n = 40
    src, tgt = ((5, 20), (5, 20)) if rule == "one_to_one" else ((0, 25), (10, 30))
    plain = build(n, src, tgt, rule, 0, **kw)
    flagged = build(n, src, tgt, rule, O.NO_AUTAPSES, **kw)
    keep = plain["source"] != plain["target"]
    assert keep.sum() < keep.size or rule == "pairwise_bernoulli"
    for k in plain:
        assert np.array_equal(flagged[k], plain[k][keep]), (rule, k)
    both = build(n, src, tgt, rule, O.NO_AUTAPSES | O.NO_MULTAPSES, **kw)  # no multapses to begin with: same result
    for k in plain:
        assert np.array_equal(both[k], flagged[k])
    if rule == "one_to_one":
        assert flagged["source"].size == 0  # identical ranges: every pair is an autapse


def test_a2_bernoulli_p1_without_autapses_is_all_to_all_minus_the_diagonal():
    a = build(30, (0, 30), (0, 30), "pairwise_bernoulli", O.NO_AUTAPSES, p=1.0)
    want = [(s, t) for s in range(30) for t in range(30) if s != t]
    assert list(zip(a["source"].tolist(), a["target"].tolist())) == want


@pytest.mark.parametrize("rule", ["fixed_indegree", "fixed_outdegree", "fixed_total_number"])
def test_a3_a4_redraw_changes_only_the_autapses(rule):
    n, K = 12, 3000
    kw = dict(degree_or_total=K if rule != "fixed_total_number" else 40000)
    plain = build(n, (0, n), (0, n), rule, 0, **kw)
    flagged = build(n, (0, n), (0, n), rule, O.NO_AUTAPSES, **kw)
    assert flagged["source"].size == plain["source"].size
    assert not np.any(flagged["source"] == flagged["target"])
    was_ok = plain["source"] != plain["target"]
    assert 0.85 < was_ok.mean() < 0.97  # about 1/12 were autapses
    for k in plain:
        assert np.array_equal(flagged[k][was_ok], plain[k][was_ok]), k
    # weight and delay never change (words 2, 3 of the attempt-0 call)
    assert np.array_equal(flagged["weight"], plain["weight"]) and np.array_equal(flagged["delay"], plain["delay"])
    # exact degrees kept
    if rule == "fixed_indegree":
        assert np.array_equal(np.bincount(flagged["target"], minlength=n), np.full(n, K))
    if rule == "fixed_outdegree":
        assert np.array_equal(np.bincount(flagged["source"], minlength=n), np.full(n, K))
    # the redrawn partners are uniform over the n - 1 allowed ones
    red = ~was_ok
    part = flagged["source" if rule != "fixed_outdegree" else "target"][red]
    fixed = flagged["target" if rule != "fixed_outdegree" else "source"][red]
    rel = (part.astype(np.int64) - fixed.astype(np.int64)) % n  # 1 .. n-1, uniform if the redraw is
    counts = np.bincount(rel, minlength=n)[1:]
    assert counts.sum() == red.sum() and chi2_ok(counts, red.sum() / (n - 1))


def test_a3_target_outside_the_sources_is_untouched():
    plain = build(50, (0, 20), (30, 10), "fixed_indegree", 0, degree_or_total=100)
    flagged = build(50, (0, 20), (30, 10), "fixed_indegree", O.NO_AUTAPSES, degree_or_total=100)
    for k in plain:
        assert np.array_equal(plain[k], flagged[k])


@pytest.mark.parametrize("rule", ["fixed_indegree", "fixed_outdegree"])
@pytest.mark.parametrize("flags", [O.NO_MULTAPSES, O.NO_MULTAPSES | O.NO_AUTAPSES])
def test_a5_partners_are_distinct_and_degrees_exact(rule, flags):
    n, K = 60, 17
    c = build(n, (0, n), (0, n), rule, flags, degree_or_total=K)
    fixed = c["target" if rule == "fixed_indegree" else "source"]
    part = c["source" if rule == "fixed_indegree" else "target"]
    assert fixed.size == n * K and np.array_equal(fixed, np.repeat(np.arange(n), K))  # creation order: i = f K + k
    for f in range(n):
        p = part[f * K:(f + 1) * K]
        assert len(set(p.tolist())) == K
        if flags & O.NO_AUTAPSES:
            assert f not in p
    # weights and delays are those of the unflagged rule (stream 0, idx i)
    plain = build(n, (0, n), (0, n), rule, 0, degree_or_total=K)
    assert np.array_equal(c["weight"], plain["weight"]) and np.array_equal(c["delay"], plain["delay"])


def test_a5_full_degree_gives_every_partner_once():
    n = 23
    c = build(n, (0, n), (0, n), "fixed_indegree", O.NO_MULTAPSES, degree_or_total=n)
    for t in range(n):
        assert sorted(c["source"][t * n:(t + 1) * n].tolist()) == list(range(n))
    c = build(n, (0, n), (0, n), "fixed_outdegree", O.NO_MULTAPSES | O.NO_AUTAPSES, degree_or_total=n - 1)
    for s in range(n):
        assert sorted(c["target"][s * (n - 1):s * (n - 1) + n - 1].tolist()) == [x for x in range(n) if x != s]


def test_a5_uniform_over_partners_and_over_ordered_pairs():
    n_src, n_tgt, K = 5, 24000, 2
    c = build(n_src + n_tgt, (0, n_src), (n_src, n_tgt), "fixed_indegree", O.NO_MULTAPSES, degree_or_total=K)
    s = c["source"].reshape(n_tgt, K)
    assert chi2_ok(np.bincount(s[:, 0], minlength=n_src), n_tgt / n_src)
    assert chi2_ok(np.bincount(s[:, 1], minlength=n_src), n_tgt / n_src)
    pair = s[:, 0].astype(np.int64) * n_src + s[:, 1]
    counts = np.bincount(pair, minlength=n_src * n_src)
    assert np.all(counts[[i * n_src + i for i in range(n_src)]] == 0)
    off = counts[[i * n_src + j for i in range(n_src) for j in range(n_src) if i != j]]
    assert chi2_ok(off, n_tgt / 20.0)
    # a larger partner set: marginal uniformity over 300 sources
    c = build(300 + 2000, (0, 300), (300, 2000), "fixed_indegree", O.NO_MULTAPSES, degree_or_total=30)
    assert chi2_ok(np.bincount(c["source"], minlength=300), 2000 * 30 / 300)


def test_explicit_node_arrays_under_the_flags():
    o = O.Oracle(dt_ms=0.1)
    o.create_population(100)
    src = np.array([7, 3, 50, 21, 99, 0], dtype=np.uint32)
    tgt = np.array([3, 4, 99, 8], dtype=np.uint32)
    o.set_rule_flags(O.NO_AUTAPSES)
    o.connect(src, tgt, R["all_to_all"], weight=W, delay_ms=D, seed=1)
    c = o.connections(sorted=False)
    got = list(zip(np.array(c["source"]).tolist(), np.array(c["target"]).tolist()))
    assert got == [(int(s), int(t)) for s in src for t in tgt if s != t]
    o.set_rule_flags(O.NO_AUTAPSES | O.NO_MULTAPSES)
    o.connect(src, tgt, R["fixed_indegree"], degree_or_total=5, weight=W, delay_ms=D, seed=2)
    c = o.connections(sorted=False)
    s2, t2 = np.array(c["source"])[len(got):], np.array(c["target"])[len(got):]
    assert np.array_equal(t2, np.repeat(tgt, 5))
    for j, t in enumerate(tgt):
        p = s2[j * 5:(j + 1) * 5].tolist()
        assert len(set(p)) == 5 and int(t) not in p and set(p) <= set(src.tolist())
        if int(t) in (3, 99):  # the target is among the sources: the five others, all of them
            assert sorted(p) == sorted(x for x in src.tolist() if x != int(t))
    # repeated ids are refused under either flag, accepted without
    dup = np.array([1, 2, 2], dtype=np.uint32)
    assert o.connect_rc(dup, tgt, R["all_to_all"], weight=W, delay_ms=D) == -1
    o.set_rule_flags(0)
    assert o.connect_rc(dup, tgt, R["all_to_all"], weight=W, delay_ms=D) == 0
    o.close()


def test_rejected_combinations():
    o = O.Oracle(dt_ms=0.1)
    o.create_population(10)
    o.set_rule_flags(O.NO_MULTAPSES)
    assert o.connect_rc((0, 10), (0, 10), R["fixed_total_number"], degree_or_total=5, weight=W, delay_ms=D) == -1  # A6
    assert o.connect_rc((0, 4), (0, 10), R["fixed_indegree"], degree_or_total=5, weight=W, delay_ms=D) == -1   # K > M
    assert o.connect_rc((0, 4), (0, 10), R["fixed_indegree"], degree_or_total=4, weight=W, delay_ms=D) == 0
    o.set_rule_flags(O.NO_MULTAPSES | O.NO_AUTAPSES)
    assert o.connect_rc((0, 4), (0, 10), R["fixed_indegree"], degree_or_total=4, weight=W, delay_ms=D) == -1   # targets 0-3 have 3
    assert o.connect_rc((0, 4), (4, 6), R["fixed_indegree"], degree_or_total=4, weight=W, delay_ms=D) == 0
    o.set_rule_flags(O.NO_AUTAPSES)
    assert o.connect_rc((2, 1), (2, 1), R["fixed_indegree"], degree_or_total=1, weight=W, delay_ms=D) == -1    # no partner
    assert o.connect_rc((2, 1), (2, 1), R["fixed_total_number"], degree_or_total=1, weight=W, delay_ms=D) == -1
    n = o.num_connections()
    assert n == 4 * 10 + 4 * 6  # the refused calls left nothing behind
    with pytest.raises(O.OracleError):
        o.set_rule_flags(4)
    o.close()


def test_flags_zero_is_the_unflagged_path():
    for rule, kw in (("fixed_indegree", dict(degree_or_total=7)), ("all_to_all", {}), ("pairwise_bernoulli", dict(p=0.2))):
        a = build(30, (0, 15), (10, 20), rule, 0, **kw)
        o = O.Oracle(dt_ms=0.1)
        o.create_population(30)
        o.connect((0, 15), (10, 20), R[rule], weight=W, delay_ms=D, seed=11, **kw)
        c = o.connections(sorted=False)
        for k in a:
            assert np.array_equal(a[k], np.array(c[k]))
        o.close()
