"""The multi-rank path of sharded construction (paper_2306_09855_b200/sharding.py; reading S1) with two CPU processes over
gloo.  The construction itself only exists as CUDA kernels, so the backend the ranks drive here is the oracle (same method
names as the binding): what is covered is the host logic -- the node partition, which shard a rank builds, that the shard
sizes gathered over the process group add up to the unsharded network, that the out-degrees reduce to the unsharded ones,
and that what rank r holds is the unsharded network filtered by what r owns."""
import os
import socket

import numpy as np
import torch.multiprocessing as mp

from paper_2306_09855_b200 import replicas, sharding, workloads as WL


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), WORLD_SIZE=str(world), RANK=str(rank),
                      LOCAL_RANK=str(rank))
    import oracle
    dist = replicas.init("gloo")
    net = WL.config2_microcircuit(scale=0.02)
    o = oracle.Oracle(dt_ms=net.dt_ms)
    sharding.build_shard(net, o, world, rank)
    c = o.connections(sorted=True)
    sizes = sharding.shard_sizes(dist, c["n"])
    outd = sharding.summed_out_degree(dist, np.array(o.degree_histogram(1)[0]))
    replicas.barrier(dist)
    out[rank] = (sizes, outd.tolist(), np.array(c["source"]).tolist(), np.array(c["target"]).tolist(), np.array(c["delay"]).tolist())
    o.close()
    dist.destroy_process_group()


def test_two_ranks_build_the_two_halves_of_the_network():
    import oracle
    world, port = 2, _free_port()
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(world, port, out), nprocs=world, join=True)
        res = dict(out)
    net = WL.config2_microcircuit(scale=0.02)
    full = oracle.Oracle(dt_ms=net.dt_ms)
    WL.run(net, full)
    fc = full.connections(sorted=True)
    fs, ft, fd = (np.array(fc[k]) for k in ("source", "target", "delay"))
    foutd = np.array(full.degree_histogram(1)[0])
    full.close()
    assert res[0][0] == res[1][0] and sum(res[0][0]) == fs.size  # every rank sees the same sizes; they add up
    assert res[0][1] == res[1][1] == foutd.tolist()
    bounds = sharding.partition(net.n_nodes, world)
    assert bounds[0] == 0 and bounds[-1] == net.n_nodes
    for r in range(world):
        own = (ft >= bounds[r]) & (ft < bounds[r + 1])
        assert res[r][0][r] == int(own.sum())
        assert res[r][2] == fs[own].tolist() and res[r][3] == ft[own].tolist() and res[r][4] == fd[own].tolist()


def test_partition_covers_every_node_once():
    for n, w in ((77169, 8), (10, 3), (5, 8), (1, 1)):
        b = sharding.partition(n, w)
        assert b[0] == 0 and b[-1] == n and all(b[i] <= b[i + 1] for i in range(w))
        assert sum(sharding.owned_range(n, w, r)[1] for r in range(w)) == n
