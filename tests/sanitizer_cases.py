"""Small end-to-end cases meant to be run UNDER compute-sanitizer (SURVEY section 4 item (4), section 5 "race detection"):

    compute-sanitizer --tool memcheck  python tests/sanitizer_cases.py
    compute-sanitizer --tool racecheck python tests/sanitizer_cases.py
    compute-sanitizer --tool synccheck python tests/sanitizer_cases.py

configs[0] and scaled configs[1] rules through every organisation variant (default, pairs, single-pass look-back, bulk-fed, bucket-first,
both COPASS modes) with the usual element-by-element comparison against the oracle, then spike delivery in its fused
(cooperative) and two-kernel forms.  Exit code 0 = every parity check held; the sanitizer's own report says whether it saw
a hazard.  profiles/r02_sanitizer.md holds the outcome.  Not collected by pytest (no test_ prefix)."""
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402


def main():
    import torch
    import oracle
    from paper_2306_09855_b200 import binding, workloads as WL
    from tests import parity_util as PU
    assert torch.cuda.is_available()
    which = sys.argv[1] if len(sys.argv) > 1 else "all"
    variants = {"default": 0, "pairs": binding.FLAG_SORT_PAIRS, "onesweep": binding.FLAG_SORT_ONESWEEP,
                "bulk": binding.FLAG_SORT_BULK, "buckets": binding.FLAG_SORT_BUCKETS, "copass": binding.FLAG_ORGANISE_COPASS,
                "copass_shift": binding.FLAG_ORGANISE_COPASS | binding.FLAG_COPASS_SHIFT}
    if which in ("all", "organise"):
        nets = [(WL.config0_tiny(), 0), (WL.config0_tiny(), 64), (WL.config0_tiny(), 10)]
        for rule in ("one_to_one", "all_to_all", "fixed_indegree", "fixed_outdegree", "fixed_total_number", "pairwise_bernoulli"):
            nets.append((WL.config1_rule(rule, scale=0.03), 4096))  # 240 + 60 nodes, several tiles and blocks
        for net, B in nets:
            for name, flags in variants.items():
                if name.startswith("copass"):
                    o = oracle.Oracle(dt_ms=net.dt_ms, block_size=B)
                    WL.run(net, o)
                    g = binding.NC(dt_ms=net.dt_ms, block_size=B, flags=flags)
                    WL.run(net, g)
                    PU.compare_sorted(g, o, net, name)
                    PU.compare_index(g.read_index(), o.index(), name)
                    g.close()
                    o.close()
                else:
                    PU.full_parity(net, oracle, binding, B=B, flags=flags)
                print(f"ok {net.name} B={B} {name}", flush=True)
    if which in ("all", "delivery"):
        for two in ("0", "1"):
            os.environ["NC_DELIVERY_TWO_KERNELS"] = two
            net = WL.config0_tiny()
            o, g = PU.build_both(net, oracle, binding)
            od, gd = oracle.Delivery(o), binding.Delivery(g, 1024)
            inp = torch.zeros(net.n_nodes, dtype=torch.float32, device="cuda")
            rng = np.random.default_rng(0)
            for k in range(50):
                nodes = rng.choice(net.n_nodes, size=7 if k < 20 else 0, replace=False).astype(np.uint32)
                want = np.zeros(net.n_nodes)
                od.step(nodes, None, want)
                inp.zero_()
                gd.step(torch.from_numpy(nodes.astype(np.int32)).cuda(), None, inp)
                assert np.abs(inp.cpu().numpy() - want).max() <= 1e-5 * max(1.0, np.abs(want).max()), f"delivery step {k}"
            assert gd.counts()["events"] == od.counts()[1]
            gd.close(); od.close(); g.close(); o.close()
            print(f"ok delivery two_kernels={two}", flush=True)
    print("sanitizer cases OK")


if __name__ == "__main__":
    main()
