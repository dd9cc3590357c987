"""B200-native construction of spiking-network connectivity (hot path of arXiv 2306.09855).

The compute path is the hand-written sm_100a CUDA library `libnc.so` (C ABI in include/nc.h); this
package is the thin ctypes binding over it (`binding`), its build step (`build`) and the synthetic
workload recipes (`workloads`).  Nothing here falls back to the CPU: if the CUDA library is missing or
no GPU is present the binding raises.
"""
__all__ = ["binding", "build", "workloads"]
