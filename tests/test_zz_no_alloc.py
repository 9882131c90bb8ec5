"""tdpd_sort_cells_noalloc (include/tdpd.h): the radix sort of row a2 with its scratch in a fixed device array of the
library, for callers that cannot allocate.  Checked, bit for bit (integer work), against the order the EXISTING path
produces: the binning a simulation runs with its workspace-carved scratch (tdpd_debug_get_binning -> sorted_id), on two
calls in a row that share the array (the second smaller, with another number of passes, explicit values and in place),
and against numpy's stable sort at the maximum size.  This file sorts last on purpose: the suite runs with pytest -x."""
import numpy as np
import pytest

import tdpd_workloads as W

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def T():
    import paper_1611_06163_b200 as T
    return T


def existing_path_order(T, w):
    """Keys and sorted order of the existing path: the particle's cell, numbered in the order the simulation's own sort
    (Morton rank of the cell, ties by previous slot = load order) put the cells, and the ids in sorted order."""
    sim = T.Simulation.from_workload(w)
    b = sim.debug_binning()
    sid = b["sorted_id"].astype(np.int64)
    c = b["cell_xyz"].astype(np.int64)
    lin = (c[:, 2] * b["ncell"][1] + c[:, 1]) * b["ncell"][0] + c[:, 0]
    seq = lin[sid]
    rank_sorted = np.r_[0, np.cumsum(np.diff(seq) != 0)]      # dense rank of the cell, along the sorted order
    keys = np.empty(len(sid), np.uint32)
    keys[sid] = rank_sorted.astype(np.uint32)                  # key of particle id
    return keys, sid.astype(np.uint32)


def dev(torch, a):
    return torch.from_numpy(np.ascontiguousarray(a).view(np.int32)).cuda()


def host(t):
    return t.cpu().numpy().view(np.uint32)


def test_noalloc_sort_matches_the_simulation_sort_twice_in_a_row(T):
    import torch
    torch.cuda.set_device(0)
    T.noalloc_init()
    st = torch.cuda.current_stream().cuda_stream

    # ---- call 1: 87,808 fluid particles, values = 0 .. n-1 (NULL), 2 passes: the result lands in the output arrays
    w1 = W.make_fluid("t", (28, 28, 28), 4.0, seed=W.BASE_SEED + 21)
    keys1, sid1 = existing_path_order(T, w1)
    n1 = len(keys1)
    assert 80000 < n1 <= T.NOALLOC_MAX_N
    bits1 = int(keys1.max()).bit_length()
    assert 8 < bits1 <= 16
    dk, ok, ov = dev(torch, keys1), torch.empty(n1, dtype=torch.int32, device="cuda"), torch.empty(n1, dtype=torch.int32, device="cuda")
    T.sort_cells_noalloc(dk.data_ptr(), 0, n1, bits1, ok.data_ptr(), ov.data_ptr(), st)
    got_k1, got_v1 = host(ok), host(ov)
    assert np.array_equal(got_v1, sid1)                        # the existing path's order, bit for bit
    assert np.array_equal(got_k1, keys1[sid1])
    assert np.array_equal(host(dk), keys1)                     # input untouched

    # ---- call 2, straight after: a smaller suspension (the scratch still holds call 1's histograms and keys),
    # 3 passes (key_bits = 20: the result passes through the scratch side an odd number of times), explicit values, in place
    w2 = W.small_suspension(seed=11, box=(20, 20, 12), n_rbc=1)
    keys2, sid2 = existing_path_order(T, w2)
    n2 = len(keys2)
    assert n2 < n1 // 4
    ids = np.arange(n2, dtype=np.uint32)
    tag = (ids * np.uint32(2654435761)) ^ np.uint32(0x9E3779B9)         # values that are not a permutation of 0..n-1
    dk2, dv2 = dev(torch, keys2), dev(torch, tag)
    T.sort_cells_noalloc(dk2.data_ptr(), dv2.data_ptr(), n2, 20, dk2.data_ptr(), dv2.data_ptr(), st)
    assert np.array_equal(host(dv2), tag[sid2])
    assert np.array_equal(host(dk2), keys2[sid2])

    # ---- call 1 again after the smaller one: same answer as before
    T.sort_cells_noalloc(dk.data_ptr(), 0, n1, bits1, ok.data_ptr(), ov.data_ptr(), st)
    assert np.array_equal(host(ov), sid1) and np.array_equal(host(ok), got_k1)

    # ---- and under stream capture, where an allocation (or any synchronising call) would invalidate the capture:
    # the call is recorded into a CUDA graph, the outputs are cleared, the graph is replayed twice
    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g, stream=side):
        T.sort_cells_noalloc(dk.data_ptr(), 0, n1, bits1, ok.data_ptr(), ov.data_ptr(), side.cuda_stream)
    for _ in range(2):
        ok.zero_(); ov.zero_()
        torch.cuda.synchronize()
        g.replay()
        torch.cuda.synchronize()
        assert np.array_equal(host(ov), sid1) and np.array_equal(host(ok), got_k1)


def test_noalloc_sort_at_the_maximum_size_and_its_limits(T):
    import torch
    torch.cuda.set_device(0)
    st = torch.cuda.current_stream().cuda_stream
    n = T.NOALLOC_MAX_N
    rng = np.random.default_rng(W.BASE_SEED + 22)
    keys = rng.integers(0, 2 ** 32, n, dtype=np.uint64).astype(np.uint32)
    keys[: n // 8] &= np.uint32(0xFF)                                   # many equal keys: stability matters
    dk = dev(torch, keys)
    ok, ov = torch.empty(n, dtype=torch.int32, device="cuda"), torch.empty(n, dtype=torch.int32, device="cuda")
    for _ in range(2):                                                  # 4 passes, full scratch, twice
        T.sort_cells_noalloc(dk.data_ptr(), 0, n, 32, ok.data_ptr(), ov.data_ptr(), st)
        order = np.argsort(keys, kind="stable")
        assert np.array_equal(host(ov), order.astype(np.uint32))
        assert np.array_equal(host(ok), keys[order])
    # a ragged size (one partial tile) and a single element
    for m in (1, 4097):
        T.sort_cells_noalloc(dk.data_ptr(), 0, m, 32, ok.data_ptr(), ov.data_ptr(), st)
        order = np.argsort(keys[:m], kind="stable")
        assert np.array_equal(host(ov)[:m], order.astype(np.uint32))
    # arrays that are only 4-byte aligned (views that start one element in), 2 and 3 passes: the sort lands in them
    for bits in (16, 24):
        m = 20000
        kin = keys[1:m + 1] & np.uint32((1 << bits) - 1)
        dk.view(torch.int32)[1:m + 1].copy_(torch.from_numpy(kin.view(np.int32)))
        T.sort_cells_noalloc(dk.data_ptr() + 4, 0, m, bits, ok.data_ptr() + 4, ov.data_ptr() + 4, st)
        order = np.argsort(kin, kind="stable")
        assert np.array_equal(host(ov)[1:m + 1], order.astype(np.uint32))
        assert np.array_equal(host(ok)[1:m + 1], kin[order])
    # beyond the maximum: a clear error, nothing enqueued, the outputs keep their contents
    before = host(ov).copy()
    with pytest.raises(T.TdpdError) as e:
        T.sort_cells_noalloc(dk.data_ptr(), 0, n + 1, 32, ok.data_ptr(), ov.data_ptr(), st)
    assert e.value.code == -1 and "TDPD_NOALLOC_MAX_N" in str(e.value) and str(n + 1) in str(e.value)
    assert np.array_equal(host(ov), before)
    for bad_bits in (0, 33):
        with pytest.raises(T.TdpdError):
            T.sort_cells_noalloc(dk.data_ptr(), 0, 16, bad_bits, ok.data_ptr(), ov.data_ptr(), st)
    with pytest.raises(T.TdpdError):
        T.sort_cells_noalloc(0, 0, 16, 8, ok.data_ptr(), ov.data_ptr(), st)
    T.sort_cells_noalloc(0, 0, 0, 8, 0, 0, st)                          # n = 0: a no-op
