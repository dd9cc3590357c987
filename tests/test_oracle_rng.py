"""Pins for the oracle's RNG layer (readings D2, D3, D5, D6): known answers, golden vectors,
closed-form properties and statistics.  CPU only."""
import math
import struct
from pathlib import Path

import numpy as np
import pytest
from scipy import stats

GOLD = Path(__file__).parent / "golden"
INF = math.inf


def _rows(name):
    for line in (GOLD / name).read_text().splitlines():
        line = line.strip()
        if line and not line.startswith("#"):
            yield line.split()


def test_philox_known_answers(oracle_mod):
    """Random123 KATs -- a wrong multiplier, round count, key bump or output order fails here."""
    n = 0
    for r in _rows("philox_kat.txt"):
        v = [int(x, 16) for x in r]
        assert oracle_mod.philox4x32_10(v[0:4], v[4:6]) == tuple(v[6:10])
        n += 1
    assert n == 3


def test_philox_counter_bijection_and_avalanche(oracle_mod):
    """For a fixed key Philox is a bijection of the 128-bit counter: distinct counters give distinct
    outputs; flipping one counter bit flips about half of the 128 output bits."""
    key = (123, 456)
    outs = {oracle_mod.philox4x32_10((i, 0, 0, 0), key) for i in range(4096)}
    assert len(outs) == 4096
    flips = []
    base = oracle_mod.philox4x32_10((77, 5, 9, 1), key)
    for word in range(4):
        for bit in range(32):
            c = [77, 5, 9, 1]
            c[word] ^= 1 << bit
            o = oracle_mod.philox4x32_10(c, key)
            flips.append(sum(bin(a ^ b).count("1") for a, b in zip(base, o)))
    assert 56 < np.mean(flips) < 72 and min(flips) > 30


def test_philox_words_uniform(oracle_mod):
    """Chi-square of the top byte of each output word over 20k calls."""
    counts = np.zeros((4, 256))
    for i in range(20000):
        o = oracle_mod.philox4x32_10((i, 0, 3, 0), (42, 0))
        for k in range(4):
            counts[k, o[k] >> 24] += 1
    for k in range(4):
        p = stats.chisquare(counts[k]).pvalue
        assert p > 1e-4, (k, p)


@pytest.mark.parametrize("n", [1, 2, 3, 7, 10, 80, 2000, 20683, 200000, 2**31 + 5, 2**32 - 1])
def test_bounded_is_floor_scaling(oracle_mod, n):
    """rand(N) as multiply-high: range [0,N), monotone, and the preimage of v is the
    interval [ceil(v 2^32/N), ceil((v+1) 2^32/N) - 1] (so bucket sizes are floor or ceil of 2^32/N)."""
    b = oracle_mod.bounded
    assert b(0, n) == 0 and b(2**32 - 1, n) == n - 1
    rng = np.random.default_rng(n % 1000)
    vs = {0, n - 1, n // 2} | {int(v) for v in rng.integers(0, n, size=50)}
    for v in vs:
        lo = -((-v * 2**32) // n)  # ceil(v 2^32 / n)
        hi = -((-(v + 1) * 2**32) // n) - 1
        assert b(lo, n) == v and b(hi, n) == v
        if lo > 0:
            assert b(lo - 1, n) == v - 1
        if hi < 2**32 - 1:
            assert b(hi + 1, n) == v + 1
        assert hi - lo + 1 in (2**32 // n, -((-2**32) // n))


def test_bounded_exhaustive_small_words(oracle_mod):
    """Brute force over a dense sweep of words for tiny N: every value hit, counts differ by <= 1 step."""
    for n in (1, 3, 5, 64):
        words = np.arange(0, 2**32, 2**16, dtype=np.uint64)  # 65536 equally spaced words
        vals = np.array([oracle_mod.bounded(int(w), n) for w in words])
        assert vals.min() == 0 and vals.max() == n - 1
        assert np.all(np.diff(vals) >= 0)
        c = np.bincount(vals, minlength=n)
        assert c.max() - c.min() <= 1


def _mv():
    for r in _rows("micro_vectors.txt"):
        yield dict(rule=r[1], seed=int(r[2]), proj=int(r[3]), s0=int(r[4]), n_src=int(r[5]), t0=int(r[6]),
                   n_tgt=int(r[7]), K=int(r[8]), w=(float(r[9]), float(r[10]), float(r[11]), float(r[12])),
                   d=(float(r[13]), float(r[14]), float(r[15]), INF), idx=int(r[16]),
                   words=[int(x, 16) for x in r[17:21]], s=int(r[21]), t=int(r[22]), whex=int(r[23], 16),
                   x=float(r[24]), steps=int(r[25]))


def test_golden_micro_vectors(oracle_mod):
    """SURVEY.md 8(c) golden micro-vectors: counter/key layout (D2), word use (D3/D4), uniforms (D5),
    Box-Muller branch assignment (D6), clamp (D7) and rounding (D8)."""
    n = 0
    for g in _mv():
        words = oracle_mod.philox4x32_10((g["idx"], 0, g["proj"], 0), (g["seed"], 0))
        assert list(words) == g["words"]
        r = oracle_mod.eval_synapse((g["s0"], g["n_src"]), (g["t0"], g["n_tgt"]), oracle_mod.FIXED_INDEGREE, g["K"], 0.0,
                                    g["w"], g["d"], g["seed"], g["proj"], 0.1, g["idx"])
        assert (r["source"], r["target"]) == (g["s"], g["t"])
        assert struct.unpack("I", struct.pack("f", r["weight"]))[0] == g["whex"]
        assert abs(r["x"] - g["x"]) < 1e-8
        assert r["delay"] == g["steps"]
        n += 1
    assert n == 7


def test_golden_misc_vectors(oracle_mod):
    rows = list(_rows("misc_vectors.txt"))
    for r in rows:
        if r[0] == "ftn":
            i, w0, w1, s, t = int(r[1]), int(r[2], 16), int(r[3], 16), int(r[4]), int(r[5])
            words = oracle_mod.philox4x32_10((i, 0, 0, 0), (7, 0))
            assert words[0] == w0 and words[1] == w1
            o = oracle_mod.eval_synapse((0, 20683), (0, 20683), oracle_mod.FIXED_TOTAL_NUMBER, 3, 0.0,
                                        (1, 0, -INF, INF), (1, 0, -INF, INF), 7, 0, 0.1, i)
            assert (o["source"], o["target"]) == (s, t)
        elif r[0] == "fod":  # pins which Philox word fixed_outdegree takes its target from (oracle.cpp, Eqs. 8-9)
            i, w0, w1, s, t, t_w0 = int(r[1]), int(r[2], 16), int(r[3], 16), int(r[4]), int(r[5]), int(r[6])
            words = oracle_mod.philox4x32_10((i, 0, 0, 0), (42, 0))
            assert words[0] == w0 and words[1] == w1
            assert (w1 * 8000) >> 32 == t and (w0 * 8000) >> 32 == t_w0 and t != t_w0  # the file is consistent with itself
            o = oracle_mod.eval_synapse((0, 8000), (0, 8000), oracle_mod.FIXED_OUTDEGREE, 1000, 0.0,
                                        (1, 0, -INF, INF), (1, 0, -INF, INF), 42, 0, 0.1, i)
            assert (o["source"], o["target"]) == (s, t)
        elif r[0] == "bern_T":
            assert oracle_mod.bernoulli_threshold(0.1) == int(r[1], 16)
        elif r[0] == "bern_words_idx2":
            want = [int(x, 16) for x in r[1:5]]
            assert [oracle_mod.bernoulli_trial_word(42, 0, q) for q in range(8, 12)] == want
            assert list(oracle_mod.philox4x32_10((2, 0, 0, 1), (42, 0))) == want
        elif r[0] == "bern_accepted_lt16":
            T = oracle_mod.bernoulli_threshold(0.1)
            assert [q for q in range(16) if oracle_mod.bernoulli_trial_word(42, 0, q) < T] == [int(r[1])]
        elif r[0] == "bern_count_lt100000":
            T = oracle_mod.bernoulli_threshold(0.1)
            assert sum(oracle_mod.bernoulli_trial_word(42, 0, q) < T for q in range(100000)) == int(r[1])


def test_bernoulli_threshold_edges(oracle_mod):
    """Q14: p = 1 -> T = 2^32 (always accept), p = 0 -> 0 (never); floor, not round."""
    assert oracle_mod.bernoulli_threshold(1.0) == 2**32
    assert oracle_mod.bernoulli_threshold(0.0) == 0
    assert oracle_mod.bernoulli_threshold(0.5) == 2**31
    assert oracle_mod.bernoulli_threshold(0.025) == math.floor(0.025 * 2**32)
    assert oracle_mod.bernoulli_threshold(2.0**-33) == 0


def test_seed_high_word_and_stream_separation(oracle_mod):
    """key = (seed lo, seed hi): seeds differing only above bit 32 differ; 64-bit idx uses ctr[1]."""
    a = oracle_mod.bernoulli_trial_word(5, 0, 0)
    b = oracle_mod.bernoulli_trial_word(5 + (1 << 32), 0, 0)
    assert a != b
    assert oracle_mod.bernoulli_trial_word(5 + (1 << 32), 0, 0) == oracle_mod.philox4x32_10((0, 0, 0, 1), (5, 1))[0]
    q = (1 << 34) + 7  # idx = q >> 2 = 2^32 + 1 -> ctr = (1, 1, proj, 1), word 3
    assert oracle_mod.bernoulli_trial_word(9, 4, q) == oracle_mod.philox4x32_10((1, 1, 4, 1), (9, 0))[3]


def test_box_muller_identities(oracle_mod):
    """D5/D6 by inversion: z0^2 + z1^2 = -2 ln u1 and atan2(z1, z0) = 2 pi u2 (mod 2 pi), with u1, u2
    rebuilt from the (KAT-pinned) Philox words; also |z| <= sqrt(48 ln 2)."""
    for i in range(0, 3000, 7):
        words = oracle_mod.philox4x32_10((i, 0, 1, 0), (99, 0))
        r = oracle_mod.eval_synapse((0, 10), (0, 10), oracle_mod.FIXED_TOTAL_NUMBER, 1, 0.0, (0, 1, -INF, INF),
                                    (0, 1, -INF, INF), 99, 1, 0.1, i)
        u1 = ((words[2] >> 8) + 1) / 2.0**24
        u2 = (words[3] >> 8) / 2.0**24
        assert 0.0 < u1 <= 1.0 and 0.0 <= u2 < 1.0
        rr = r["z0"] ** 2 + r["z1"] ** 2
        assert abs(rr - (-2.0 * math.log(u1))) < 1e-9
        if rr > 1e-12:
            ang = math.atan2(r["z1"], r["z0"]) % (2 * math.pi)
            d = abs(ang - 2 * math.pi * u2)
            assert min(d, 2 * math.pi - d) < 1e-7
        assert abs(r["z0"]) <= math.sqrt(48 * math.log(2)) + 1e-12
        # weight = mean + sd z0 with mean 0, sd 1 and no clamp -> fp32(z0)
        assert r["weight"] == np.float32(r["z0"])


def test_normals_are_standard_normal(oracle_mod):
    """z0 and z1: mean 0, sd 1, uncorrelated; chi-square on 64 equal-probability bins."""
    o = oracle_mod.Oracle(dt_ms=1.0)
    o.create_population(1000)
    n = 400_000
    # weight = z0 exactly; delay path is checked elsewhere.  z1 via a second projection trick is not
    # needed: eval_synapse exposes both.
    o.connect((0, 1000), (0, 1000), oracle_mod.FIXED_TOTAL_NUMBER, degree_or_total=n, weight=(0.0, 1.0, -INF, INF),
              delay_ms=(1.0, 0.0, -INF, INF), seed=2024)
    z0 = o.connections()["weight"].astype(np.float64)
    assert abs(z0.mean()) < 5 / math.sqrt(n)
    assert abs(z0.std() - 1.0) < 5 / math.sqrt(2 * n)
    edges = stats.norm.ppf(np.linspace(0, 1, 65)[1:-1])
    c = np.bincount(np.searchsorted(edges, z0), minlength=64)
    assert stats.chisquare(c).pvalue > 1e-4
    z1 = np.array([oracle_mod.eval_synapse((0, 10), (0, 10), oracle_mod.FIXED_TOTAL_NUMBER, 1, 0.0, (0, 1, -INF, INF),
                                           (0, 1, -INF, INF), 2024, 0, 1.0, i)["z1"] for i in range(40000)])
    c1 = np.bincount(np.searchsorted(edges, z1), minlength=64)
    assert stats.chisquare(c1).pvalue > 1e-4
    assert abs(np.corrcoef(z0[:40000], z1)[0, 1]) < 4 / math.sqrt(40000)
