"""Pins for the oracle's rule expansion, block accounting, transforms and error behaviour
(readings D1, D4, D7-D9; Eqs. 1-13): closed forms, the paper's worked example, exact
invariants, chi-square and binomial statistics, brute force.  CPU only."""
import math
from pathlib import Path

import numpy as np
import pytest
from scipy import stats

GOLD = Path(__file__).parent / "golden"
INF = math.inf
W = (20.0, 2.0, 0.0, INF)
D = (1.5, 0.75, 0.1, INF)


def mk(oracle_mod, pops, dt=0.1, B=0):
    o = oracle_mod.Oracle(dt_ms=dt, block_size=B)
    firsts = [o.create_population(n) for n in pops]
    return o, firsts


def test_population_ids_contiguous(oracle_mod):
    """D1."""
    o, f = mk(oracle_mod, [80, 20, 7])
    assert f == [0, 80, 100] and o.num_nodes() == 107


def test_fig1_worked_example(oracle_mod):
    """PAPER.md:51 (Fig. 1): all_to_all 4x3 with B = 10 after 14 earlier connections: i -> (s,t) by
    Eqs. 6-7, positions 14..25 straddle block 1 (6 slots) and block 2 (6 slots); Eq. 1 block counts."""
    o, (a, b, c) = mk(oracle_mod, [14, 4, 3], B=10)
    o.connect((a, 14), (a, 14), oracle_mod.ONE_TO_ONE, weight=W, delay_ms=D, seed=1)
    assert o.num_connections() == 14 and o.num_blocks() == 2
    o.connect((b, 4), (c, 3), oracle_mod.ALL_TO_ALL, weight=W, delay_ms=D, seed=1)
    assert o.num_connections() == 26 and o.num_blocks() == 3
    conn = o.connections()
    rows = [l.split() for l in (GOLD / "fig1_all_to_all.txt").read_text().splitlines() if l and l[0] != "#"]
    assert len(rows) == 12
    for i, ds, dt in rows:
        pos = 14 + int(i)
        assert conn["source"][pos] == b + int(ds) and conn["target"][pos] == c + int(dt)
    blocks = [o.block_slot(14 + i)[0] for i in range(12)]
    assert blocks == [1] * 6 + [2] * 6  # N_prevconns,2 = 6 (Eq. 3)
    assert [o.block_slot(14 + i)[1] for i in range(12)] == [4, 5, 6, 7, 8, 9, 0, 1, 2, 3, 4, 5]


@pytest.mark.parametrize("B", [1, 7, 10, 64, 4096])
def test_eq1_block_count_brute_force(oracle_mod, B):
    """Eq. 1: after every call N_blocks = ceil(N_conns / B); pos -> (block, slot) bijective."""
    o, (a,) = mk(oracle_mod, [50], B=B)
    rng = np.random.default_rng(B)
    total = 0
    for call in range(12):
        n = int(rng.integers(0, 40))
        o.connect((a, 50), (a, 50), oracle_mod.FIXED_TOTAL_NUMBER, degree_or_total=n, weight=W, delay_ms=D, seed=call)
        total += n
        assert o.num_connections() == total
        assert o.num_blocks() == -(-total // B)
    seen = set()
    for pos in range(total):
        blk, slot = o.block_slot(pos)
        assert 0 <= slot < B and blk < o.num_blocks() and blk * B + slot == pos
        seen.add((blk, slot))
    assert len(seen) == total


def test_one_to_one_and_all_to_all_closed_form(oracle_mod):
    """Eqs. 4-7 with non-zero s0, t0."""
    o, (a, b, c) = mk(oracle_mod, [5, 37, 37])
    o.connect((b, 37), (c, 37), oracle_mod.ONE_TO_ONE, weight=W, delay_ms=D, seed=3)
    o.connect((a, 5), (b, 37), oracle_mod.ALL_TO_ALL, weight=W, delay_ms=D, seed=3)
    conn = o.connections()
    i = np.arange(37)
    assert np.array_equal(conn["source"][:37], b + i) and np.array_equal(conn["target"][:37], c + i)
    i = np.arange(5 * 37)
    assert np.array_equal(conn["source"][37:], a + i // 37) and np.array_equal(conn["target"][37:], b + i % 37)
    assert conn["n"] == 37 + 5 * 37


def test_fixed_indegree_invariants(oracle_mod):
    """Eqs. 10-11: t = t0 + floor(i/K) exactly, every target has in-degree K, N =
    N_targets K; sources uniform on the source range (chi-square); out-degree ~ Binomial(N, 1/N_src)."""
    n_src, n_tgt, K = 300, 500, 400
    o, (a, b) = mk(oracle_mod, [n_src, n_tgt])
    o.connect((a, n_src), (b, n_tgt), oracle_mod.FIXED_INDEGREE, degree_or_total=K, weight=W, delay_ms=D, seed=11)
    conn = o.connections()
    n = n_tgt * K
    assert conn["n"] == n
    assert np.array_equal(conn["target"], b + np.arange(n) // K)
    indeg, mx = o.degree_histogram(0)
    assert np.all(indeg[b:b + n_tgt] == K) and np.all(indeg[:b] == 0) and mx == K
    s = conn["source"].astype(np.int64) - a
    assert s.min() >= 0 and s.max() < n_src
    outdeg = np.bincount(s, minlength=n_src)
    assert stats.chisquare(outdeg).pvalue > 1e-4
    assert abs(outdeg.var() / (n * (1 / n_src) * (1 - 1 / n_src)) - 1) < 0.3
    od, _ = o.degree_histogram(1)
    assert np.array_equal(od[a:a + n_src], outdeg)


def test_fixed_outdegree_invariants(oracle_mod):
    """Eqs. 8-9."""
    n_src, n_tgt, K = 400, 250, 300
    o, (a, b) = mk(oracle_mod, [n_src, n_tgt])
    o.connect((a, n_src), (b, n_tgt), oracle_mod.FIXED_OUTDEGREE, degree_or_total=K, weight=W, delay_ms=D, seed=12)
    conn = o.connections()
    n = n_src * K
    assert conn["n"] == n
    assert np.array_equal(conn["source"], a + np.arange(n) // K)
    t = conn["target"].astype(np.int64) - b
    assert t.min() >= 0 and t.max() < n_tgt
    assert stats.chisquare(np.bincount(t, minlength=n_tgt)).pvalue > 1e-4
    outdeg, mx = o.degree_histogram(1)
    assert np.all(outdeg[a:a + n_src] == K) and mx == K


def test_fixed_total_number_invariants(oracle_mod):
    """Eqs. 12-13, Q3: exactly N i.i.d. pairs; marginals uniform; s and t independent
    (chi-square on a coarse 2-D grid)."""
    n_src, n_tgt, N = 640, 480, 300_000
    o, (a, b) = mk(oracle_mod, [n_src, n_tgt])
    o.connect((a, n_src), (b, n_tgt), oracle_mod.FIXED_TOTAL_NUMBER, degree_or_total=N, weight=W, delay_ms=D, seed=13)
    conn = o.connections()
    assert conn["n"] == N
    s = conn["source"].astype(np.int64) - a
    t = conn["target"].astype(np.int64) - b
    assert 0 <= s.min() and s.max() < n_src and 0 <= t.min() and t.max() < n_tgt
    assert stats.chisquare(np.bincount(s, minlength=n_src)).pvalue > 1e-4
    assert stats.chisquare(np.bincount(t, minlength=n_tgt)).pvalue > 1e-4
    grid = np.zeros((16, 16))
    np.add.at(grid, (s * 16 // n_src, t * 16 // n_tgt), 1)
    assert stats.chi2_contingency(grid)[1] > 1e-4


def test_pairwise_bernoulli_invariants(oracle_mod):
    """Q13/Q14: each ordered pair tried once; count ~ Binomial(N_src N_tgt, T/2^32); in-degree ~
    Binomial(N_src, p); no duplicate pair; ascending q; p = 1 == all_to_all pairs; p = 0 empty."""
    n_src, n_tgt, p = 400, 300, 0.1
    o, (a, b) = mk(oracle_mod, [n_src, n_tgt])
    o.connect((a, n_src), (b, n_tgt), oracle_mod.PAIRWISE_BERNOULLI, p=p, weight=W, delay_ms=D, seed=14)
    conn = o.connections()
    pe = oracle_mod.bernoulli_threshold(p) / 2.0**32
    n_pairs = n_src * n_tgt
    assert abs(conn["n"] - n_pairs * pe) < 5 * math.sqrt(n_pairs * pe * (1 - pe))
    q = (conn["source"].astype(np.int64) - a) * n_tgt + (conn["target"].astype(np.int64) - b)
    assert np.all(np.diff(q) > 0)  # ascending and duplicate-free
    indeg = np.bincount(conn["target"] - b, minlength=n_tgt)
    ks = np.arange(0, n_src + 1)
    pmf = stats.binom.pmf(ks, n_src, pe)
    lo, hi = np.searchsorted(np.cumsum(pmf), [0.01, 0.99])
    obs = np.bincount(np.clip(indeg, lo, hi), minlength=hi + 1)[lo:hi + 1]
    exp = pmf[lo:hi + 1].copy()
    exp[0] += pmf[:lo].sum()
    exp[-1] += pmf[hi + 1:].sum()
    assert stats.chisquare(obs, exp * n_tgt / exp.sum()).pvalue > 1e-4
    # acceptance is exactly "trial word < T"
    T = oracle_mod.bernoulli_threshold(p)
    acc = [qq for qq in range(2000) if oracle_mod.bernoulli_trial_word(14, 0, qq) < T]
    assert list(q[q < 2000]) == acc
    # p = 1 and p = 0
    o1, (a1, b1) = mk(oracle_mod, [7, 5])
    o1.connect((a1, 7), (b1, 5), oracle_mod.PAIRWISE_BERNOULLI, p=1.0, weight=W, delay_ms=D, seed=3)
    o1.connect((a1, 7), (b1, 5), oracle_mod.PAIRWISE_BERNOULLI, p=0.0, weight=W, delay_ms=D, seed=3)
    c1 = o1.connections()
    i = np.arange(35)
    assert c1["n"] == 35 and np.array_equal(c1["source"], a1 + i // 5) and np.array_equal(c1["target"], b1 + i % 5)


def test_bernoulli_p1_equals_all_to_all_synapses(oracle_mod):
    """The synapse stream is indexed by q, so with p = 1 weights and delays equal those of all_to_all
    issued as the same projection id."""
    oa, (a, b) = mk(oracle_mod, [9, 11])
    oa.connect((a, 9), (b, 11), oracle_mod.ALL_TO_ALL, weight=W, delay_ms=D, seed=5)
    ob, _ = mk(oracle_mod, [9, 11])
    ob.connect((a, 9), (b, 11), oracle_mod.PAIRWISE_BERNOULLI, p=1.0, weight=W, delay_ms=D, seed=5)
    ca, cb = oa.connections(), ob.connections()
    for k in ("source", "target", "weight", "delay"):
        assert np.array_equal(ca[k], cb[k])


def test_projection_id_and_seed_decorrelate(oracle_mod):
    o, (a,) = mk(oracle_mod, [1000])
    for seed in (1, 1, 2):
        o.connect((a, 1000), (a, 1000), oracle_mod.FIXED_TOTAL_NUMBER, degree_or_total=5000, weight=W, delay_ms=D, seed=seed)
    s = o.connections()["source"].reshape(3, 5000)
    assert not np.array_equal(s[0], s[1]) and not np.array_equal(s[1], s[2])
    assert abs(np.corrcoef(s[0], s[1])[0, 1]) < 0.08


def test_weight_distribution(oracle_mod):
    """D7: mean/sd within 5 standard errors, chi-square on 64 equal-probability bins, sign clip, sd = 0."""
    n = 400_000
    o, (a,) = mk(oracle_mod, [100])
    o.connect((a, 100), (a, 100), oracle_mod.FIXED_TOTAL_NUMBER, degree_or_total=n, weight=(-80.0, 8.0, -INF, 0.0),
              delay_ms=D, seed=21)
    w = o.connections()["weight"].astype(np.float64)
    assert np.all(w <= 0)
    assert abs(w.mean() + 80.0) < 5 * 8 / math.sqrt(n) and abs(w.std() - 8.0) < 5 * 8 / math.sqrt(2 * n)
    edges = stats.norm.ppf(np.linspace(0, 1, 65)[1:-1], loc=-80.0, scale=8.0)
    assert stats.chisquare(np.bincount(np.searchsorted(edges, w), minlength=64)).pvalue > 1e-4
    # heavy clipping: mean 1, sd 2, lo 0 -> P(w == 0) = Phi(-0.5)
    o2, (a2,) = mk(oracle_mod, [100])
    o2.connect((a2, 100), (a2, 100), oracle_mod.FIXED_TOTAL_NUMBER, degree_or_total=100_000, weight=(1.0, 2.0, 0.0, 2.5),
               delay_ms=D, seed=22)
    w2 = o2.connections()["weight"]
    assert w2.min() == 0.0 and w2.max() == 2.5
    for val, pr in ((0.0, stats.norm.cdf(-0.5)), (2.5, 1 - stats.norm.cdf(0.75))):
        frac = np.mean(w2 == val)
        assert abs(frac - pr) < 5 * math.sqrt(pr * (1 - pr) / 100_000)
    # sd = 0 -> constant ("identical values for all connections")
    o3, (a3,) = mk(oracle_mod, [10])
    o3.connect((a3, 10), (a3, 10), oracle_mod.ALL_TO_ALL, weight=(3.25, 0.0, -INF, INF), delay_ms=(0.7, 0.0, -INF, INF), seed=1)
    c3 = o3.connections()
    assert np.all(c3["weight"] == np.float32(3.25)) and np.all(c3["delay"] == 7)


def test_delay_distribution(oracle_mod):
    """D8: steps = round(d/dt) >= 1.  Histogram against the discretised clipped normal
    P(k) = Phi(((k+.5)dt - mu)/sd) - Phi(((k-.5)dt - mu)/sd) (k >= 2), P(1) = Phi((1.5 dt - mu)/sd);
    a floor instead of round, a missing clamp or a wrong dt shifts this visibly.  Weight and delay share
    one Box-Muller pair but are uncorrelated."""
    n = 400_000
    mu, sd, dt = 1.5, 0.75, 0.1
    o, (a,) = mk(oracle_mod, [100], dt=dt)
    o.connect((a, 100), (a, 100), oracle_mod.FIXED_TOTAL_NUMBER, degree_or_total=n, weight=W, delay_ms=(mu, sd, 0.1, INF), seed=31)
    c = o.connections()
    d = c["delay"].astype(np.int64)
    assert d.min() == 1 and d.max() <= math.floor((mu + 5.769 * sd) / dt + 0.5)
    kmax = 45
    ks = np.arange(1, kmax + 1)
    cdf = lambda v: stats.norm.cdf((v - mu) / sd)  # noqa: E731
    P = cdf((ks + 0.5) * dt) - cdf((ks - 0.5) * dt)
    P[0] = cdf(1.5 * dt)
    P[-1] = 1.0 - cdf((kmax - 0.5) * dt)
    obs = np.bincount(np.minimum(d, kmax), minlength=kmax + 1)[1:]
    assert stats.chisquare(obs, P * n).pvalue > 1e-4
    assert abs(obs[0] / n - stats.norm.cdf(-1.8)) < 5 * math.sqrt(0.036 * 0.964 / n)  # ~3.6 %
    assert abs(np.corrcoef(c["weight"], d)[0, 1]) < 4 / math.sqrt(n)
    # another resolution and an upper clip
    o2, (a2,) = mk(oracle_mod, [100], dt=0.25)
    o2.connect((a2, 100), (a2, 100), oracle_mod.FIXED_TOTAL_NUMBER, degree_or_total=50_000, weight=W,
               delay_ms=(1.0, 1.0, 0.1, 2.0), seed=32)
    d2 = o2.connections()["delay"]
    assert d2.min() == 1 and d2.max() == 8
    assert abs(np.mean(d2 == 8) - (1 - stats.norm.cdf(0.875))) < 5 * math.sqrt(0.19 * 0.81 / 50_000)


def test_delay_rounding_half_up_exact_cases(oracle_mod):
    """Q5: constants land exactly: 0.25 ms / 0.1 ms = 2.5 -> 3 (half up); 0.24 -> 2; below one step -> 1."""
    for ms, dt, want in ((0.25, 0.1, 3), (0.24, 0.1, 2), (0.01, 0.1, 1), (0.75, 0.5, 2), (1.25, 0.5, 3), (6553.5, 0.1, 65535)):
        o, (a,) = mk(oracle_mod, [4], dt=dt)
        o.connect((a, 4), (a, 4), oracle_mod.ONE_TO_ONE, weight=W, delay_ms=(ms, 0.0, -INF, INF), seed=1)
        assert set(o.connections()["delay"].tolist()) == {want}, (ms, dt)


def test_error_behaviour(oracle_mod):
    """SURVEY.md 8(b) conventions: invalid arguments, state and capacity errors; a failed connect leaves
    the context unchanged and does not consume a projection id."""
    E = oracle_mod
    o, (a, b) = mk(oracle_mod, [10, 20])
    ok = dict(weight=W, delay_ms=D, seed=1)
    assert o.connect_rc((a, 10), (b, 20), E.ONE_TO_ONE, **ok) == E.ERR_INVALID_ARG  # N_src != N_tgt
    assert o.connect_rc((25, 10), (b, 20), E.ALL_TO_ALL, **ok) == E.ERR_INVALID_ARG  # outside created nodes
    assert o.connect_rc((a, 0), (b, 20), E.ALL_TO_ALL, **ok) == E.ERR_INVALID_ARG
    assert o.connect_rc((a, 10), (b, 20), E.PAIRWISE_BERNOULLI, p=1.5, **ok) == E.ERR_INVALID_ARG
    assert o.connect_rc((a, 10), (b, 20), E.PAIRWISE_BERNOULLI, p=-0.1, **ok) == E.ERR_INVALID_ARG
    assert o.connect_rc((a, 10), (b, 20), 9, **ok) == E.ERR_INVALID_ARG
    assert o.connect_rc((a, 10), (b, 20), E.ALL_TO_ALL, weight=(1, -1, -INF, INF), delay_ms=D, seed=1) == E.ERR_INVALID_ARG
    assert o.connect_rc((a, 10), (b, 20), E.ALL_TO_ALL, weight=(1, 1, 2.0, 1.0), delay_ms=D, seed=1) == E.ERR_INVALID_ARG
    assert o.connect_rc((a, 10), (b, 20), E.ALL_TO_ALL, weight=W, delay_ms=(7000.0, 0.0, -INF, INF), seed=1) == E.ERR_CAPACITY
    assert o.connect_rc((a, 10), (b, 20), E.FIXED_TOTAL_NUMBER, degree_or_total=2**32, **ok) == E.ERR_CAPACITY
    assert o.connect_rc((a, 10), (b, 20), E.FIXED_INDEGREE, degree_or_total=2**31, **ok) == E.ERR_CAPACITY
    assert o.num_connections() == 0
    # projection id not consumed by failures: next success is projection 0
    o.connect((a, 10), (b, 20), E.FIXED_TOTAL_NUMBER, degree_or_total=5, **ok)
    ref = [E.eval_synapse((a, 10), (b, 20), E.FIXED_TOTAL_NUMBER, 5, 0, W, D, 1, 0, 0.1, i)["source"] for i in range(5)]
    assert o.connections()["source"].tolist() == ref
    o.finalize()
    assert o.connect_rc((a, 10), (b, 20), E.ALL_TO_ALL, **ok) == E.ERR_STATE
    with pytest.raises(E.OracleError):
        o.finalize()
    with pytest.raises(E.OracleError):
        E.Oracle(dt_ms=0.0)
    # degree 0 is legal and yields nothing
    o2, (a2,) = mk(oracle_mod, [5])
    o2.connect((a2, 5), (a2, 5), E.FIXED_INDEGREE, degree_or_total=0, **ok)
    assert o2.num_connections() == 0
