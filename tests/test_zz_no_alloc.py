"""nc_index_static (include/nc_static.h) against the index nc_finalize builds.

Why the entry point exists: some users of the library cannot allocate device memory at the moment they need an index --
a simulation loop with a latency budget (cudaMalloc / cudaFree make the whole device wait), a process whose own pool
already owns the card (a library's cudaMalloc just fails), code that may only touch the buffers and the stream it was
given.  nc_index_static therefore takes its scratch from an array inside the library image, of fixed size (so n is
limited), shared by every call on the device (so calls must not overlap on the GPU, and the array still holds what the
last call wrote).

What is checked here, bit for bit (integer outputs: the tolerance of every index test in this suite is zero):
  - on the organised source / delay arrays of a finalized context, nc_index_static fills the caller's buffers with the
    same src_offsets, group_ptr, group_count, group_start, group_delay and group total as nc_read_index returns;
  - on two calls in a row without any wait in between -- first a network of many tiles, then a smaller one, whose
    status words the first call left non-zero -- and on a third call over the first network again;
  - the second and third call do not change the device's free memory (nothing was allocated behind the caller's back);
  - a size beyond NC_INDEX_STATIC_MAX_CONNECTIONS is refused with NC_ERR_CAPACITY and a message, and too small a group
    capacity is reported in *d_error while everything that fits is still right.
The file name sorts last on purpose: pytest -x stops at the first failure, and a failure here must not hide the
parity tests.  It needs nothing from the tests before it (it passes alone in a fresh process as well)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def _build(net, binding, WL):
    g = binding.NC(dt_ms=net.dt_ms)
    WL.run(net, g)  # creates the populations, connects every projection, nc_finalize
    return g


class _Buffers:
    """Everything nc_index_static writes, allocated by the CALLER (here: torch) before the calls."""

    def __init__(self, torch, n_nodes, capacity):
        i32 = dict(dtype=torch.int32, device="cuda")
        self.src_offsets = torch.full((n_nodes + 1,), -1, **i32)
        self.group_ptr = torch.full((n_nodes + 1,), -1, **i32)
        self.group_count = torch.full((n_nodes,), -1, **i32)
        self.group_start = torch.full((max(capacity, 1),), -1, **i32)
        self.group_delay = torch.full((max(capacity, 1),), -1, dtype=torch.int16, device="cuda")
        self.total = torch.full((1,), -1, **i32)
        self.error = torch.full((1,), -1, **i32)
        self.capacity = capacity

    def call(self, binding, view, n, n_nodes):
        binding.index_static(view.source, view.delay, n, n_nodes, self.src_offsets.data_ptr(), self.group_ptr.data_ptr(),
                             self.group_count.data_ptr(), self.group_start.data_ptr(), self.group_delay.data_ptr(),
                             self.capacity, self.total.data_ptr(), self.error.data_ptr())

    def check(self, want, what, expect_error=0):
        G = want["total_groups"]
        u32 = lambda t: t.cpu().numpy().view(np.uint32)
        assert int(self.error.item()) == expect_error, f"{what}: d_error = {int(self.error.item())}"
        assert int(self.total.item()) == G, f"{what}: total groups {int(self.total.item())} != {G}"
        for name in ("src_offsets", "group_ptr", "group_count"):
            assert np.array_equal(u32(getattr(self, name)), want[name]), f"{what}: {name} differs from nc_read_index"
        k = min(G, self.capacity)
        assert np.array_equal(u32(self.group_start)[:k], want["group_start"][:k]), f"{what}: group_start differs"
        assert np.array_equal(self.group_delay.cpu().numpy().view(np.uint16)[:k], want["group_delay"][:k]), f"{what}: group_delay differs"
        if self.capacity > k:  # nothing written behind the last group
            assert (self.group_start[k:self.capacity] == -1).all() and (self.group_delay[k:self.capacity] == -1).all(), what


def test_index_without_allocation_equals_the_allocating_path_on_consecutive_calls():
    import torch
    from paper_2306_09855_b200 import binding, build, workloads as WL
    build.build()
    torch.cuda.set_device(0)
    big = WL.config2_microcircuit(scale=0.05)  # ~7.5e5 connections over 3,858 nodes: some 46 tiles of 16,384 and a ragged tail
    small = WL.config0_tiny()                  # less than one tile
    gb, gs = _build(big, binding, WL), _build(small, binding, WL)
    try:
        want_b, want_s = gb.read_index(), gs.read_index()
        vb, vs = gb.get_connections(sorted=True), gs.get_connections(sorted=True)
        nb, ns = gb.num_connections(), gs.num_connections()
        assert nb > 20 * 16384 and 0 < ns < 16384
        # the caller sizes the group arrays: the exact total is known here; the second set is sized by the general bound n
        b1 = _Buffers(torch, big.n_nodes, want_b["total_groups"])
        s1 = _Buffers(torch, small.n_nodes, ns)
        b2 = _Buffers(torch, big.n_nodes, nb)
        # set-up call (first call on the device: looks up the scratch array's address), as a user would make it at start-up
        warm = _Buffers(torch, small.n_nodes, 0)
        binding.index_static(None, None, 0, small.n_nodes, warm.src_offsets.data_ptr(), warm.group_ptr.data_ptr(),
                             warm.group_count.data_ptr(), None, None, 0, warm.total.data_ptr(), warm.error.data_ptr())
        torch.cuda.synchronize()
        assert int(warm.total.item()) == 0 and int(warm.error.item()) == 0
        assert not warm.src_offsets.any() and not warm.group_ptr.any() and not warm.group_count.any()

        b1.call(binding, vb, nb, big.n_nodes)
        torch.cuda.synchronize()
        free_before = torch.cuda.mem_get_info()[0]
        # two calls in a row on one stream, nothing waited for in between: the second starts from the first one's leftovers
        s1.call(binding, vs, ns, small.n_nodes)
        b2.call(binding, vb, nb, big.n_nodes)
        torch.cuda.synchronize()
        free_after = torch.cuda.mem_get_info()[0]
        b1.check(want_b, "first call, 46 tiles")
        s1.check(want_s, "second call, one tile after 46")
        b2.check(want_b, "third call, 46 tiles after one")
        assert free_after == free_before, f"device memory changed across the calls: {free_before} -> {free_after} bytes free"
        print(f"nc_index_static: {nb} and {ns} connections, {want_b['total_groups']} and {want_s['total_groups']} groups, "
              f"three calls bit-exact against nc_read_index; free device memory unchanged ({free_after} B)")
    finally:
        gb.close()
        gs.close()


def test_index_without_allocation_refuses_what_does_not_fit():
    import torch
    from paper_2306_09855_b200 import binding, build, workloads as WL
    build.build()
    torch.cuda.set_device(0)
    net = WL.config0_tiny()
    g = _build(net, binding, WL)
    try:
        want, v, n = g.read_index(), g.get_connections(sorted=True), g.num_connections()
        G = want["total_groups"]
        assert G > 8
        # beyond the size the built-in scratch array was made for: refused before anything is enqueued
        buf = _Buffers(torch, net.n_nodes, G)
        with pytest.raises(binding.NCError) as e:
            binding.index_static(v.source, v.delay, binding.INDEX_STATIC_MAX_CONNECTIONS + 1, net.n_nodes,
                                 buf.src_offsets.data_ptr(), buf.group_ptr.data_ptr(), buf.group_count.data_ptr(),
                                 buf.group_start.data_ptr(), buf.group_delay.data_ptr(), G, buf.total.data_ptr(),
                                 buf.error.data_ptr())
        assert e.value.code == binding.ERR_CAPACITY and "NC_INDEX_STATIC_MAX_CONNECTIONS" in str(e.value)
        torch.cuda.synchronize()
        assert int(buf.total.item()) == -1 and (buf.src_offsets == -1).all(), "a refused call must not touch the outputs"
        # a misaligned input array is an argument error
        with pytest.raises(binding.NCError) as e:
            binding.index_static(v.source + 4, v.delay, n - 1, net.n_nodes, buf.src_offsets.data_ptr(),
                                 buf.group_ptr.data_ptr(), None, buf.group_start.data_ptr(), buf.group_delay.data_ptr(), G,
                                 buf.total.data_ptr(), buf.error.data_ptr())
        assert e.value.code == binding.ERR_INVALID_ARG
        # group arrays too small: flagged on the device; the groups that fit and every per-node array are still right
        tight = _Buffers(torch, net.n_nodes, G - 5)
        tight.call(binding, v, n, net.n_nodes)
        torch.cuda.synchronize()
        tight.check(want, "capacity five short", expect_error=binding.INDEX_STATIC_GROUPS)
        # and the very next call with room for everything is clean again
        buf.call(binding, v, n, net.n_nodes)
        torch.cuda.synchronize()
        buf.check(want, "after the flagged call")
    finally:
        g.close()
