"""More connections than one context's 32-bit positions can count, on ONE B200 (the paper's
largest network has ~10^9 connections, N = 10^6 with K = 10^4 did not fit its 40 GB card).  A context holds at most
2^32 - 1 connections; a larger network is built as shards (nc_set_shard), each with its own positions: here 100,000 nodes,
four fixed_indegree calls of 1.25e9 connections each = 5.0e9 connections > 2^32, as two shards by target (1.875e9 and
3.125e9 connections), organised inside the storage blocks (COPASS, 21 B per connection), the larger one 66 GB.

Checked per shard: the exact count; the whole organised order, a chunk at a time (keys ascend, ties in creation order,
out-degrees, group heads, every index array equal to its definition); and sampled connections against the oracle's
per-synapse function through the permutation (a shard's creation position p is the p-th connection it owns, which for
fixed_indegree with a contiguous owned target range is call c, index i = first owned index of c + (p - start of c))."""
import math

import numpy as np
import pytest

from paper_2306_09855_b200 import workloads as WL

pytestmark = pytest.mark.gpu
INF = math.inf
N, K, CALLS = 100_000, 50_000, 4
W, D = (20.0, 2.0, 0.0, INF), (1.5, 0.75, 0.1, INF)
PER = N // CALLS  # targets per call


@pytest.fixture(scope="module")
def nc_mod():
    from paper_2306_09855_b200 import binding, build
    build.build()
    return binding


def _build_shard(nc_mod, first, count):
    g = nc_mod.NC(dt_ms=0.1, flags=nc_mod.FLAG_ORGANISE_COPASS)
    g.create_population(N)
    g.set_shard(first, count)
    for c in range(CALLS):
        g.connect((0, N), (c * PER, PER), WL.RULE_IDS["fixed_indegree"], degree_or_total=K, weight=W, delay_ms=D, seed=2306)
    return g


@pytest.mark.parametrize("shard", [(0, 37_500), (37_500, 62_500)])
def test_five_billion_connections_as_two_shards(nc_mod, oracle_mod, shard):
    import torch
    free, _ = torch.cuda.mem_get_info()
    if free < 110 * 2**30:
        pytest.skip("needs ~100 GB of free device memory")
    first, count = shard
    g = _build_shard(nc_mod, first, count)
    # what the shard owns of every call: targets [lo, hi) of the call -> indexes [lo K, hi K)
    own = []
    for c in range(CALLS):
        lo = min(max(first - c * PER, 0), PER)
        hi = min(max(first + count - c * PER, 0), PER)
        own.append((lo * K, hi * K))
    starts = np.concatenate([[0], np.cumsum([b - a for a, b in own])]).astype(np.int64)
    n = int(starts[-1])
    assert CALLS * PER * K > 2**32 and g.num_connections() == n == count * K
    g.finalize()
    st = g.stats()
    assert st["n_blocks"] == (n + (1 << 24) - 1) >> 24
    idx = g.read_index()
    rng = np.random.default_rng(first)
    out_deg = np.zeros(N, dtype=np.int64)
    gcount = np.zeros(N, dtype=np.int64)
    heads, head_delay = [], []
    prev_key = prev_perm = None
    checked = mism = 0
    chunk = 1 << 26
    for j0 in range(0, n, chunk):
        cnt = min(chunk, n - j0)
        s = g.read_connections(sorted=True, first=j0, count=cnt)
        key = (s["source"].astype(np.uint64) << np.uint64(16)) | s["delay"].astype(np.uint64)
        perm = s["perm"]
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
        out_deg += np.bincount(s["source"], minlength=N)
        gcount += np.bincount(s["source"][h - j0], minlength=N)
        prev_key, prev_perm = key[-1], perm[-1]
        # sampled connections of this chunk against the oracle, through the permutation
        pick = rng.integers(0, cnt, size=4000)
        p = s["perm"][pick].astype(np.int64)
        call = np.searchsorted(starts, p, side="right") - 1
        for c in np.unique(call):
            m = call == c
            i = own[c][0] + (p[m] - starts[c])
            o = oracle_mod.eval_synapses((0, N), (c * PER, PER), WL.RULE_IDS["fixed_indegree"], K, 0.0, W, D, 2306, int(c), 0.1, i)
            assert np.array_equal(o["source"], s["source"][pick][m]) and np.array_equal(o["target"], s["target"][pick][m])
            assert np.all(np.abs(o["weight"].astype(np.float64) - s["weight"][pick][m]) <= 1e-5 * 22.0)
            dd = o["delay"].astype(np.int64) - s["delay"][pick][m].astype(np.int64)
            bad = dd != 0
            assert np.all(np.abs(dd[bad]) == 1) and np.all(o["boundary"][bad] == 1)
            mism += int(bad.sum())
            checked += int(m.sum())
        del s
    assert mism <= math.ceil(1e-7 * checked), (mism, checked)
    heads = np.concatenate(heads)
    assert idx["total_groups"] == heads.size
    assert np.array_equal(idx["group_start"], heads) and np.array_equal(idx["group_delay"], np.concatenate(head_delay))
    assert np.array_equal(idx["src_offsets"], np.concatenate([[0], np.cumsum(out_deg)]).astype(np.uint32))
    assert np.array_equal(idx["group_count"], gcount.astype(np.uint32))
    assert np.array_equal(idx["group_ptr"], np.concatenate([[0], np.cumsum(gcount)]).astype(np.uint32))
    print(f"shard {shard}: {n} connections, {st['n_blocks']} blocks, peak {st['bytes_peak'] / 2**30:.1f} GiB, "
          f"{checked} sampled against the oracle, {mism} boundary mismatches")
    g.close()
