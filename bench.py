#!/usr/bin/env python
"""bench.py -- synapses constructed per second (generate + sort + index), device-timed, on the
cortical-microcircuit-shaped workload (BASELINE.json configs[2]: 77,169 neurons, 298,880,970 synapses).

    python bench.py --gpus N --steps K --warmup W            # the CUDA path (one replica per GPU)
    python bench.py --impl reference --steps K --warmup W    # the CPU oracle on a bounded sample

One "step" = one pass of the whole hot path: create the populations, issue all 55 nc_connect calls (rule
expansion + draws + append into block storage), nc_finalize (per-pass digit counts and scans, record-carrying digit passes, index).
Prints ONE JSON line on rank 0.  See DESIGN.md "Measurement" for how every field is obtained.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "synapses constructed/s (generate+sort+index, device-timed)"
UNIT = "synapses/s"
# algorithmic bytes per synapse
# sort_pass: the record-carrying digit pass reads 16 B and writes 16 B per synapse (SURVEY 8(d) "carry (tgt, w) as extra
# payload -> P x 32 B, permute vanishes"); histogram: 6 B (first pass) + 1 B per later pass; index: 6 B read twice.
BYTES = {"generate": 14, "histogram": 8, "sort_pass": 32, "permute": 26, "index": 12}


TRAFFIC_FILE = os.path.join("profiles", "r03_scatter_traffic.txt")
KERNEL_FILE = os.path.join("paper_2306_09855_b200", "csrc", "nc_sort_split.cuh")


def kernel_file_sha256():
    import hashlib
    return hashlib.sha256(open(os.path.join(ROOT, KERNEL_FILE), "rb").read()).hexdigest()


def ncu_traffic_per_launch():
    """(dram__bytes_read.sum + dram__bytes_write.sum of one middle scatter pass, where it was captured, stale?) from the
    committed ncu --set full capture.  The figure is a property of the kernel source: the file records the SHA-256 of
    nc_sort_split.cuh as it was when ncu ran, and the figure is only reported while the shipped file still has that hash
    (the GPU box has no .git, so a content hash and not a commit id); otherwise traffic is null and traffic_stale true."""
    out, where, sha = None, None, None
    try:
        for line in open(os.path.join(ROOT, TRAFFIC_FILE)):
            if line.startswith("traffic_bytes_per_launch"):
                out = float(line.split("=")[1])
            if line.startswith("captured_at"):
                where = line.split("=", 1)[1].strip()
            if line.startswith("kernel_file_sha256"):
                sha = line.split("=", 1)[1].strip()
    except Exception:
        pass
    stale = out is None or sha is None or sha != kernel_file_sha256()
    return (None if stale else out), where, stale


def workload(name: str):
    from paper_2306_09855_b200 import workloads as WL
    if name == "c2":
        return WL.config2_microcircuit()
    if name.startswith("c2x"):
        return WL.config2_microcircuit(scale=float(name[3:]))
    if name == "c3":
        return WL.config3_large_indegree()
    if name == "c4":
        return WL.config4_large_bernoulli()
    if name.startswith("c1:"):
        return WL.config1_rule(name[3:])
    if name == "c0":
        return WL.config0_tiny()
    raise SystemExit(f"unknown workload {name}")


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""

    def __init__(self, index: int):
        super().__init__(daemon=True)
        self.index, self.samples, self.reasons, self.max_mhz, self._halt = index, [], set(), None, threading.Event()
        self.ready = threading.Event()  # NVML is initialised: sampling has begun

    def run(self):
        try:
            import pynvml as nv
            nv.nvmlInit()
            h = nv.nvmlDeviceGetHandleByIndex(self.index)
            self.max_mhz = nv.nvmlDeviceGetMaxClockInfo(h, nv.NVML_CLOCK_SM)
            names = {
                nv.nvmlClocksThrottleReasonHwSlowdown: "hw_slowdown",
                nv.nvmlClocksThrottleReasonHwThermalSlowdown: "hw_thermal_slowdown",
                nv.nvmlClocksThrottleReasonSwThermalSlowdown: "sw_thermal_slowdown",
                nv.nvmlClocksThrottleReasonSwPowerCap: "sw_power_cap",
            }
            self.ready.set()
            while not self._halt.is_set():
                self.samples.append(nv.nvmlDeviceGetClockInfo(h, nv.NVML_CLOCK_SM))
                r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(h)
                for bit, nm in names.items():
                    if r & bit:
                        self.reasons.add(nm)
                time.sleep(0.004)
        except Exception as e:  # NVML missing: report that instead of failing the bench
            self.reasons.add(f"nvml_unavailable:{type(e).__name__}")
            self.ready.set()

    def stop(self):
        self._halt.set()
        self.join(timeout=2)
        return {"sm_mhz": statistics.median(self.samples) if self.samples else None, "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(self.samples)}


BLOCK_SIZE = 0  # --block-size: connections per storage block (0 = the library's default 2^24)


SHARD = None  # --sharded: (world, rank)


def one_step(binding, WL, net, flags):
    """The public API call sequence a user makes.  Returns the (still open) context."""
    g = binding.NC(dt_ms=net.dt_ms, flags=flags, block_size=BLOCK_SIZE)
    if SHARD is not None:
        from paper_2306_09855_b200 import sharding
        sharding.build_shard(net, g, *SHARD)
    else:
        WL.run(net, g)
    return g


def cpu_model():
    try:
        for line in open("/proc/cpuinfo"):
            if line.startswith("model name"):
                return line.split(":", 1)[1].strip()
    except Exception:
        pass
    return "unknown"


PHASE_SPLIT = {}  # filled by cpu_oracle_sample: seconds of the last step's generate / sort + index


def cpu_oracle_sample(sample_scale: float, steps: int = 1):
    """The oracle as it stands, one thread pinned to one core, on a bounded sample of the same workload.
    generate = the connect calls, organise = oc_finalize (stable sort + index)."""
    import oracle
    from paper_2306_09855_b200 import workloads as WL
    net = WL.config2_microcircuit(scale=sample_scale)
    oracle.build()
    old_aff = None
    try:
        old_aff = os.sched_getaffinity(0)
        os.sched_setaffinity(0, {sorted(old_aff)[-1]})
    except Exception:
        old_aff = None
    times, n = [], 0
    try:
        for _ in range(steps):
            t0 = time.perf_counter()
            o = oracle.Oracle(dt_ms=net.dt_ms)
            WL.run(net, o, finalize=False)
            t1 = time.perf_counter()
            o.finalize()
            t2 = time.perf_counter()
            n = o.num_connections()
            times.append(t2 - t0)
            PHASE_SPLIT.update(generate_s=t1 - t0, sort_index_s=t2 - t1)
            o.close()
    finally:
        if old_aff is not None:
            os.sched_setaffinity(0, old_aff)
    return net, n, times


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    scale = args.sample_scale if args.sample_scale else 0.1
    for _ in range(args.warmup):
        cpu_oracle_sample(min(scale, 0.03))
    net, n, times = cpu_oracle_sample(scale, steps=args.steps)
    value = n * len(times) / sum(times)
    sample = f"configs[2] with populations scaled x{scale:g} ({net.n_nodes} nodes, {n} synapses, 55 projections) per step"
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * sum(times) / len(times), "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": "configs[2] cortical-microcircuit-shaped, fixed_total_number, seed 7 (bounded sample)",
                   "sample": sample},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample,
                         "phases_s": {k: round(v, 2) for k, v in PHASE_SPLIT.items()},
                         "pinned": "one thread on one core (sched_setaffinity)", "cpu_model": cpu_model(), "host_cpus": os.cpu_count()},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


def run_delivery(args):
    """Secondary measurement (not the headline metric): spike delivery over the organised
    configs[2] network, `--workload delivery:<spike probability per node per step>` (default 0.01).  One step = one
    nc_delivery_step on a seeded synthetic raster resident in HBM."""
    import numpy as np
    import torch
    from paper_2306_09855_b200 import binding, build, workloads as WL
    build.build()
    torch.cuda.set_device(0)
    rate = float(args.workload.split(":")[1]) if ":" in args.workload else 0.01
    net = WL.config2_microcircuit()
    g = binding.NC(dt_ms=net.dt_ms, flags=args.flags, block_size=args.block_size)  # --flags 16: over COPASS-organised blocks
    WL.run(net, g)
    n_nodes, n_syn = g.num_nodes(), g.num_connections()
    rng = np.random.default_rng(2306)
    total_steps = args.warmup + args.steps
    counts = rng.binomial(n_nodes, rate, size=total_steps)
    offs = np.concatenate([[0], np.cumsum(counts)])
    nodes = np.concatenate([rng.choice(n_nodes, size=int(k), replace=False) for k in counts]).astype(np.int32)
    d_nodes = torch.from_numpy(nodes).cuda()
    inp = torch.zeros(n_nodes, dtype=torch.float32, device="cuda")
    d = binding.Delivery(g, capacity=int(rate * n_nodes * 80 * 1.5) + 4096)
    stream = torch.cuda.current_stream()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    d.run(d_nodes, None, offs[:args.warmup + 1], inp)  # warm-up steps
    events0 = d.counts()["events"]
    torch.cuda.synchronize()
    ev0.record(stream)
    d.run(d_nodes, None, offs[args.warmup:], inp)      # the timed steps: one C call, one launch per step
    ev1.record(stream)
    torch.cuda.synchronize()
    c = d.counts()
    ms = ev0.elapsed_time(ev1)
    events = c["events"] - events0
    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        pass
    peak = float(peaks.get("hbm_gbs", 6650.0))
    gbs = events * 8 / (ms * 1e-3) / 1e9  # target (4 B) + weight (4 B) read per delivered connection
    line = {"metric": "synaptic events delivered/s (spike delivery over the built index, device-timed)",
            "value": events / (ms * 1e-3), "unit": "events/s", "n_gpus": 1, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32", "data": "synthetic",
            "config": {"workload": f"delivery over configs[2] ({n_nodes} nodes, {n_syn} connections), Bernoulli({rate}) "
                                   "spikes per node per step, raster resident in HBM",
                       "events_per_step": events / args.steps, "spikes_per_step": float(counts[args.warmup:].mean()),
                       "buffered_at_end": c["buffered"], "dropped": c["dropped"], "flags": args.flags},
            "gpu_launches": args.steps * (2 if os.environ.get("NC_DELIVERY_TWO_KERNELS", "0") not in ("", "0") else 1),
            "roofline": {"bound": "hbm", "kernel": "fused_step_kernel, delivery phase (8 B read per delivered connection + one fp32 atomic add)",
                         "achieved": gbs, "peak": peak, "unit": "GB/s", "frac": gbs / peak, "traffic": None}}
    print(json.dumps(line))
    d.close()
    g.close()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="nc", choices=["nc", "reference"])
    ap.add_argument("--workload", default="c2")
    ap.add_argument("--sample-scale", type=float, default=0.0, help="cpu baseline sample: population scale of configs[2]")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--flags", type=int, default=0, help="extra NC_FLAG_* bits (e.g. 4 = sort (key, position) pairs + gather; "
                    "16 = COPASS organisation inside the storage blocks, 48 = the same with the shift of Fig. 6E)")
    ap.add_argument("--block-size", type=int, default=0, help="connections per storage block B (0 = 2^24)")
    ap.add_argument("--sharded", action="store_true", help="strong scaling: the ranks build the shards of ONE network "
                    "(nc_set_shard: rank r keeps the connections whose target it owns) instead of one replica each")
    args = ap.parse_args()
    global BLOCK_SIZE
    BLOCK_SIZE = args.block_size
    if args.impl == "reference":
        return run_reference(args)
    if args.workload.startswith("delivery"):
        return run_delivery(args)

    import torch
    from paper_2306_09855_b200 import binding, build, replicas, workloads as WL
    build.build()
    world, rank, local = replicas.env_world()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (the path has no CPU fallback)")
    torch.cuda.set_device(local)
    dist = replicas.init("nccl", torch.device("cuda", local))

    def barrier():
        replicas.barrier(dist, torch.cuda.synchronize)

    net = workload(args.workload)
    stream = torch.cuda.current_stream()
    flags = binding.FLAG_TIMING | args.flags
    if args.sharded:
        global SHARD
        SHARD = (world, rank)

    # ---- warm-up (also warms torch's caching allocator: the timed steps allocate from its cache) ----
    n_syn = 0
    cold_ms = None
    for w in range(max(args.warmup, 0)):
        t0 = time.perf_counter()
        g = one_step(binding, WL, net, flags)
        n_syn = g.num_connections()
        g.synchronize()
        if w == 0:  # the one cold step: device allocations come from the driver, not from torch's cache
            cold_ms = 1e3 * (time.perf_counter() - t0)
        g.close()
    barrier()

    # ---- timed region: K steps, CUDA events on the stream the kernels are launched on ----
    sampler = ClockSampler(local)
    sampler.start()
    sampler.ready.wait(timeout=10)
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    phase_acc, launches, stats = {}, 0, {}
    barrier()
    ev0.record(stream)
    step_marks = [ev0]
    for _ in range(args.steps):
        g = one_step(binding, WL, net, flags)
        n_syn = g.num_connections()
        t = g.timings()  # synchronises this context's stream; the events were recorded on the device
        stats = g.stats()
        if flags & binding.FLAG_ORGANISE_COPASS:
            stats["copass"] = g.copass_stats()
        launches += stats["kernel_launches"]
        for k, v in t.items():
            phase_acc[k] = phase_acc.get(k, 0.0) + v
        g.close()
        step_marks.append(torch.cuda.Event(enable_timing=True))
        step_marks[-1].record(stream)
    ev1.record(stream)
    barrier()
    total_ms = ev0.elapsed_time(ev1)
    step_ms = [a.elapsed_time(b) for a, b in zip(step_marks[:-1], step_marks[1:])]
    clocks = sampler.stop()
    total_ms = replicas.max_over_ranks(dist, total_ms, "cuda")
    ms_per_step = total_ms / args.steps
    value = replicas.whole_job_rate(n_syn, args.steps, world, total_ms)
    if args.sharded:  # the ranks hold one network between them: its size is the sum of the shards
        from paper_2306_09855_b200 import sharding
        n_total = sum(sharding.shard_sizes(dist, n_syn, "cuda"))
        value = n_total * args.steps / (total_ms * 1e-3)

    # ---- end to end through the public API with host buffers: context creation, host descriptors in,
    #      index arrays read back into host memory, wall clock ----
    e2e_times, d2h = [], 0
    for _ in range(max(2, min(args.steps, 5))):
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        g = one_step(binding, WL, net, args.flags)
        idx = g.read_index()
        cnt = g.num_connections()
        g.synchronize()
        e2e_times.append(time.perf_counter() - t0)
        d2h = sum(v.nbytes for v in idx.values() if hasattr(v, "nbytes")) + 8 + 4
        nblocks = g.stats()["n_blocks"]
        g.close()
    h2d = len(net.projections) * (8 + 8 + 16 + 64 + 8) + 8 * nblocks  # per nc_connect: ranges, rule params, syn spec, seed; block table
    e2e_t = replicas.max_over_ranks(dist, statistics.median(e2e_times), "cuda")
    e2e_value = replicas.whole_job_rate(cnt, 1, world, e2e_t * 1e3)

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        pass
    peak = float(peaks.get("hbm_gbs", 6650.0))
    peak_kind = "measured (MEASURED_PEAKS.json hbm_gbs)" if "hbm_gbs" in peaks else "fallback 6.65 TB/s"
    K = args.steps
    per = {k: v / K for k, v in phase_acc.items()}
    passes = max(1, int(round(per.get("sort_passes", 0))))
    pass_ms = per["sort_pass_ms"] / passes if per.get("sort_pass_ms") else None
    roof = None
    copass = bool(flags & binding.FLAG_ORGANISE_COPASS)
    if copass and per.get("sort_pass_ms"):
        # every record goes through the digit passes twice: when its block is sorted, and in the auxiliary array
        P = max(1, int(stats.get("sort_passes") or 1))
        ach = BYTES["sort_pass"] * 2 * P * n_syn / (per["sort_pass_ms"] * 1e-3) / 1e9
        roof = {"bound": "hbm", "kernel": "scatter_pass_kernel over one block at a time (COPASS organisation: 2 x "
                                          f"{P} digit passes per connection, 16 B read + 16 B written each)",
                "achieved": ach, "peak": peak, "unit": "GB/s", "frac": ach / peak, "traffic": None,
                "peak_kind": peak_kind, "launch_ms": pass_ms, "launches_per_step": passes}
        passes = 2 * P
    elif pass_ms:
        ach = BYTES["sort_pass"] * n_syn / (pass_ms * 1e-3) / 1e9
        # the ncu figure belongs to the default path on configs[2]; stale = the kernel file changed since it was captured
        traffic = ncu_traffic_per_launch() if args.workload == "c2" and not args.flags else (None, None, None)
        roof = {"bound": "hbm", "kernel": "scatter_pass_kernel (one digit pass carrying the whole connection: 16 B read + "
                                          "16 B written per synapse)",
                "achieved": ach, "peak": peak, "unit": "GB/s", "frac": ach / peak,
                "traffic": traffic[0], "traffic_captured_at": traffic[1], "traffic_stale": traffic[2],
                "peak_kind": peak_kind,
                "launch_ms": pass_ms, "launches_per_step": passes,
                "context": "peak is a streaming copy; the pass writes ~256-byte runs that start inside 32-byte sectors, and a "
                           "copy kernel with that write pattern and no ranking reaches 5050-5390 GB/s on a B200 "
                           "(tests/cuda/membench.cu `pattern`, profiles/r02_scatter.md); the SM side of the pass (7.9 us per "
                           "tile of 4096 records, 296 tiles in flight) sits at the same rate even with the records in the L2 "
                           "(profiles/r02_buckets.md)"}
    phases = {}
    for name, b in (("generate", BYTES["generate"]), ("histogram", BYTES["histogram"]), ("sort", BYTES["sort_pass"] * passes),
                    ("permute", BYTES["permute"]), ("index", BYTES["index"])):
        ms = per.get(f"{name}_ms", 0.0)
        if ms > 0:
            gbs = b * n_syn / (ms * 1e-3) / 1e9
            phases[name] = {"ms": round(ms, 4), "alg_bytes_per_synapse": b, "GBps": round(gbs, 1),
                            "frac_of_measured_peak": round(gbs / peak, 4), "frac_of_8TBps": round(gbs / 8000.0, 4)}

    if per.get("copass_ms", 0.0) > 0:
        # COPASS organisation (Fig. 6 C-E): partitions plus the record moves (16 B read + 16 B written
        # each).  Default: gather of every output block + emptying one block into the holes; with NC_FLAG_COPASS_SHIFT
        # the left partitions and every record still to the right of the block, per output block.
        cst = stats.get("copass", {})
        moved = int(cst.get("records_moved", 0))
        gbs = 32 * moved / (per["copass_ms"] * 1e-3) / 1e9
        phases["copass_partitions_and_moves"] = {
            "ms": round(per["copass_ms"], 4), "records_moved": moved, "blocks": int(cst.get("n_blocks", 0)),
            "partitions": int(cst.get("partitions", 0)), "partition_iterations": int(cst.get("iterations", 0)),
            "aux_bytes": int(cst.get("aux_bytes", 0)),
            "mode": "shift (Fig. 6E)" if flags & binding.FLAG_COPASS_SHIFT else "hole filling",
            "alg_bytes_per_record_moved": 32, "GBps": round(gbs, 1), "frac_of_measured_peak": round(gbs / peak, 4)}
    cpu = None
    if not args.no_cpu_baseline and args.workload.startswith("c2"):
        scale = args.sample_scale if args.sample_scale else 1.0  # the bench's own inputs: all of configs[2] (~90 s on one core)
        snet, sn, st = cpu_oracle_sample(scale)
        cpu = {"value": sn / st[0], "unit": UNIT, "cores": 1, "kind": "oracle",
               "sample": f"configs[2] with populations scaled x{scale:g}: {snet.n_nodes} nodes, {sn} synapses, generate+sort+index, {st[0]:.1f} s",
               "phases_s": {k: round(v, 2) for k, v in PHASE_SPLIT.items()},
               "pinned": "one thread on one core (sched_setaffinity)", "cpu_model": cpu_model(), "host_cpus": os.cpu_count()}

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_per_step, "ms_per_step_sd": statistics.pstdev(step_ms) if len(step_ms) > 1 else 0.0,
        "cold_first_step_ms": cold_ms, "higher_is_better": True, "scaling": "strong" if args.sharded else "weak",
        "vs_baseline": None, "dtype": "u32+f32",
        "data": "synthetic",
        "config": {"workload": f"{net.name}: BASELINE.json configs[2] cortical-microcircuit-shaped network, "
                               f"{net.n_nodes} nodes, {len(net.projections)} fixed_total_number projections, seed 7"
                   if args.workload == "c2" else net.name,
                   "synapses_per_step": n_syn,
                   "parallelism": (f"one network in {world} shards by target node (nc_set_shard), no data-path collective; every "
                                   "rank generates the FULL call of the random-target rules and filters it (redundant generation: "
                                   "that part does not shrink with the number of ranks); never measured on more than one GPU"
                                   if args.sharded else "replicas only (one independent network per GPU)"),
                   "l2": "every step regenerates and re-sorts its own 4.2 GB of connections (>> 126 MB L2); no input is reused",
                   "key_bits": stats.get("key_bits"), "sort_passes": stats.get("sort_passes"), "flags": flags,
                   "block_size": args.block_size or (1 << 24), "device_bytes_peak": stats.get("bytes_peak")},
        "clocks": clocks, "gpu_launches": launches,
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                "what": "wall clock of nc_create + populations + all nc_connect + nc_finalize + nc_read_index into host buffers"},
        "roofline": roof, "phases": phases, "cpu_baseline": cpu,
    }
    print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
