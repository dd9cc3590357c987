"""Pins of the COPASS oracle (oracle/copass.cpp; Appendix A) against things other than itself:
hand-worked iterations (tests/golden/copass_partition.txt), the conditions A6-A8 by brute force, the first m elements
of a stable merge written with numpy, Eq. A3, the intermediate picture of Fig. 6, and numpy's stable argsort."""
from pathlib import Path

import numpy as np
import pytest

import oracle

GOLDEN = Path(__file__).parent / "golden" / "copass_partition.txt"


def _flatten(subs):
    lens = np.array([len(s) for s in subs], dtype=np.uint64)
    start = np.concatenate([[0], np.cumsum(lens)[:-1]]).astype(np.uint64)
    keys = np.concatenate([np.asarray(s, dtype=np.int64) for s in subs]) if lens.sum() else np.zeros(0, np.int64)
    return keys, start, lens


def _stable_merge_left_sizes(subs, m):
    """Plain definition: order every element by (value, subarray, position) and count, per subarray, how many of the
    first m it owns."""
    val = np.concatenate([np.asarray(s, dtype=np.int64) for s in subs])
    sub = np.concatenate([np.full(len(s), i) for i, s in enumerate(subs)])
    pos = np.concatenate([np.arange(len(s)) for s in subs])
    order = np.lexsort((pos, sub, val))[:m]
    return np.bincount(sub[order], minlength=len(subs))


def test_golden_hand_worked_cases():
    cases = [l for l in GOLDEN.read_text().splitlines() if l and not l.startswith("#")]
    assert len(cases) == 3
    for line in cases:
        name, subs, m, want, t, it, last = [f.strip() for f in line.split("|")]
        subs = [[int(x) for x in s.split()] for s in subs.split(";")]
        keys, start, lens = _flatten(subs)
        m_i, got_t, got_it, got_last = oracle.copass_partition(keys, start, lens, int(m))
        assert m_i.tolist() == [int(x) for x in want.split()], name
        assert (got_t, got_it, got_last) == (int(t), int(it), int(last)), name


@pytest.mark.parametrize("seed", range(12))
def test_partition_conditions_a6_a8_and_stable_merge(seed):
    rng = np.random.default_rng(seed)
    k = int(rng.integers(1, 9))
    span = int(rng.choice([2, 5, 50, 10**6]))  # few distinct values -> long runs of ties (Sec. A4)
    subs = [np.sort(rng.integers(-span, span, size=int(rng.integers(0, 40)))) for _ in range(k)]
    total = sum(len(s) for s in subs)
    if total < 2:
        subs[0] = np.array([0, 1])
        total = sum(len(s) for s in subs)
    keys, start, lens = _flatten(subs)
    for m in sorted(set([1, total - 1] + rng.integers(1, total, size=6).tolist())):
        m_i, t, it, last = oracle.copass_partition(keys, start, lens, m)
        assert int(m_i.sum()) == m                                    # A8
        for s, mi in zip(subs, m_i.astype(int)):
            assert mi <= len(s)
            assert np.all(s[:mi] <= t) and np.all(s[mi:] >= t)        # A6, A7
        assert m_i.astype(int).tolist() == _stable_merge_left_sizes(subs, m).tolist()  # readings C3, C4
        assert last in (1, 2)


def test_partition_both_last_steps_are_reached():
    rng = np.random.default_rng(5)
    seen = set()
    for _ in range(200):
        subs = [np.sort(rng.integers(0, 30, size=int(rng.integers(1, 12)))) for _ in range(4)]
        keys, start, lens = _flatten(subs)
        total = int(lens.sum())
        seen.add(oracle.copass_partition(keys, start, lens, int(rng.integers(1, total)))[3])
    assert seen == {1, 2}


def test_partition_rejects_bad_arguments():
    keys, start, lens = _flatten([[1, 2, 3], [4, 5]])
    for m in (0, 5, 6):  # 0 < m < sum N_i (reading C1)
        with pytest.raises(oracle.OracleError):
            oracle.copass_partition(keys, start, lens, m)
    keys, start, lens = _flatten([[3, 2, 1], [4, 5]])  # not ascending (A5)
    with pytest.raises(oracle.OracleError):
        oracle.copass_partition(keys, start, lens, 2)


def test_partition_iterations_grow_like_a_bisection():
    # every iteration halves the widest open interval and narrows all others with the same threshold: for subarrays
    # drawn alike the count stays near log2(N_i), far below N_i
    rng = np.random.default_rng(1)
    subs = [np.sort(rng.integers(0, 2**40, size=4096)) for _ in range(8)]
    keys, start, lens = _flatten(subs)
    _, _, it, _ = oracle.copass_partition(keys, start, lens, 4096)
    assert 8 <= it <= 60


@pytest.mark.parametrize("seed", range(10))
def test_block_sort_is_the_stable_sort_of_the_whole_array(seed):
    rng = np.random.default_rng(100 + seed)
    k = int(rng.integers(1, 8))
    sizes = rng.integers(0, 50, size=k).astype(np.uint64)
    if seed % 3 == 0:
        sizes[:] = 16  # equal blocks, as the connection blocks are
    n = int(sizes.sum())
    span = int(rng.choice([1, 3, 20, 10**9]))
    keys = rng.integers(0, span, size=n).astype(np.int64)
    vals = np.arange(n, dtype=np.uint32)
    ks, vs, _, _, st = oracle.copass_block_sort(keys, vals, sizes)
    order = np.argsort(keys, kind="stable")
    assert np.array_equal(ks, keys[order])
    assert np.array_equal(vs, order.astype(np.uint32))  # equal keys keep their original order (reading C6)
    if n:
        assert st["aux_peak"] == int(sizes.max())        # Eq. A3
    assert st["partitions"] == st["last_step_1"] + st["last_step_2"]


def test_block_sort_special_inputs():
    for keys in (np.arange(64), np.arange(64)[::-1], np.zeros(64), np.repeat(np.arange(8), 8)[::-1]):
        keys = np.asarray(keys, dtype=np.int64)
        ks, vs, _, _, st = oracle.copass_block_sort(keys, np.arange(64, dtype=np.uint32), [10] * 6 + [4])
        order = np.argsort(keys, kind="stable")
        assert np.array_equal(ks, keys[order]) and np.array_equal(vs, order.astype(np.uint32))
    # all keys equal: every partition ends with t~ equal to that value in its first iteration (Sec. A4)
    assert st["last_step_1"] + st["last_step_2"] == st["partitions"]


def test_block_sort_intermediate_state_matches_fig6():
    """After e extractions (Fig. 6 C-F repeated e times): the first e blocks are final; what is left consists of k
    ascending logical subarrays packed behind them, none of whose elements is smaller than an extracted one."""
    rng = np.random.default_rng(7)
    sizes = np.array([12, 12, 12, 12, 7], dtype=np.uint64)
    n = int(sizes.sum())
    keys = rng.integers(0, 25, size=n).astype(np.int64)
    vals = np.arange(n, dtype=np.uint32)
    final = np.sort(keys, kind="stable")
    for e in range(1, 5):
        ks, vs, sub_start, sub_len, _ = oracle.copass_block_sort(keys, vals, sizes, max_extract=e)
        done = int(sizes[:e].sum())
        assert np.array_equal(ks[:done], final[:done])
        assert np.array_equal(np.sort(ks[done:]), final[done:])  # nothing lost, nothing duplicated
        assert np.array_equal(keys[vs], ks)                      # values travelled with their keys
        assert int(sub_len.sum()) == n - done
        at = done
        for s, l in zip(sub_start.astype(int), sub_len.astype(int)):
            assert s == at                                       # packed in subarray order
            assert np.all(np.diff(ks[s:s + l]) >= 0)             # each still ascending (A5)
            at += l
        if done < n:
            assert ks[done:].min() >= ks[:done].max()
