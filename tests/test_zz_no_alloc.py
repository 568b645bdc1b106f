"""tpc_scan_exclusive_static: the prefix sum for callers that must not allocate device memory.

Some users of this library run where cudaMalloc is off limits: inside an online framework that reserved all GPU
memory at start-up and hands its components nothing but input and output buffers, or on a latency-bound path where the
device-wide stall of cudaMalloc / cudaFree is not acceptable.  For them the library's prefix-sum kernel can be run with
its scratch words (tile counter + one status word per 2048 elements) in an array built into the library instead of in
the tracker's cudaMalloc'ed work space.  This file checks that entry point against the allocating path the tracker uses
(`tpc_debug_scan_exclusive`: same kernel, scratch from cudaMalloc) -- bit-exact, as for every integer result in this
repo -- and against numpy's cumsum, on two calls in a row that share the built-in array.

The file is named so that pytest collects it LAST: with `pytest -x` a failure here cannot hide another test.  It does
not depend on what ran before it: it passes alone in a fresh process (where its first call is the one that looks up the
array's device address) and after the other GPU tests (where the library is already loaded and the array may hold
anything)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def tr():
    import torch
    assert torch.cuda.is_available(), "these tests need a CUDA device"
    torch.cuda.set_device(0)
    from paper_1712_09416_b200 import tracker
    return tracker


def counts(n, seed):
    """Seeded bin-count-like input: small non-negative int32, many zeros (empty bins), no overflow at the maximum n."""
    rng = np.random.default_rng(seed)
    a = rng.integers(0, 100, size=n, dtype=np.int32)
    a[rng.random(n) < 0.3] = 0
    return a


def expected(a):
    out = np.zeros(a.size + 1, dtype=np.int64)
    np.cumsum(a, out=out[1:])
    return out.astype(np.int32)


def run_pair(tr, sizes, seed):
    """Two calls in a row on ONE stream, no synchronisation between them (the second starts on the scratch words the
    first one left behind), each compared with the allocating path and with numpy."""
    import torch
    stream = torch.cuda.Stream()
    ins = [torch.from_numpy(counts(n, seed + k)).cuda() for k, n in enumerate(sizes)]
    outs = [torch.full((n + 1,), -7, dtype=torch.int32, device="cuda") for n in sizes]
    refs = [torch.full((n + 1,), -9, dtype=torch.int32, device="cuda") for n in sizes]
    torch.cuda.synchronize()
    for a, o in zip(ins, outs):
        tr.tpc_scan_exclusive_static(a.data_ptr(), a.numel(), o.data_ptr(), stream.cuda_stream)
    stream.synchronize()
    for a, r in zip(ins, refs):
        tr.tpc_debug_scan_exclusive(a.data_ptr(), a.numel(), r.data_ptr())
    torch.cuda.synchronize()
    for a, o, r in zip(ins, outs, refs):
        got, ref = o.cpu().numpy(), r.cpu().numpy()
        assert np.array_equal(got, ref), (a.numel(), int(np.flatnonzero(got != ref)[0]))
        assert np.array_equal(got, expected(a.cpu().numpy())), a.numel()


@pytest.mark.parametrize("sizes", [
    (1_000_003, 5_000),          # many tiles with a ragged tail, then few: stale status words of the first call remain
    (2_049, 2_048),              # around one tile
    (1, 0),                      # the degenerate cases: out = [0, a0] and out = [0]
    (5 * 36 * 159, 16 * 36 * 159),   # bins of a 5- and a 16-event batch (events x sectors x pad rows)
])
def test_static_scratch_scan_equals_the_allocating_path_twice_in_a_row(tr, sizes):
    run_pair(tr, sizes, seed=20171209)


def test_static_scratch_scan_at_its_maximum_size_and_again_after_it(tr):
    n = tr.SCAN_STATIC_MAX_N
    run_pair(tr, (n, n - 2047), seed=7)


def test_static_scratch_scan_rejects_sizes_beyond_its_array(tr):
    import torch
    n = tr.SCAN_STATIC_MAX_N + 1
    a = torch.zeros(n, dtype=torch.int32, device="cuda")
    o = torch.full((n + 1,), -7, dtype=torch.int32, device="cuda")
    with pytest.raises(tr.TpcError) as ei:
        tr.tpc_scan_exclusive_static(a.data_ptr(), n, o.data_ptr())
    assert ei.value.status == tr.TPC_ERR_CAPACITY and "TPC_SCAN_STATIC_MAX_N" in str(ei.value)
    torch.cuda.synchronize()
    assert int((o != -7).sum()) == 0            # nothing was launched
    for bad in (lambda: tr.tpc_scan_exclusive_static(a.data_ptr(), -1, o.data_ptr()),
                lambda: tr.tpc_scan_exclusive_static(None, 5, o.data_ptr()),
                lambda: tr.tpc_scan_exclusive_static(a.data_ptr(), 5, None)):
        with pytest.raises(tr.TpcError) as ei:
            bad()
        assert ei.value.status == tr.TPC_ERR_ARG
    # the limit itself is served, and a refused call leaves the entry point usable
    run_pair(tr, (4_097, 3), seed=11)


def test_static_scratch_scan_takes_no_device_memory(tr):
    """After the first call on the device (which may load the library's device code), further calls leave the amount
    of free device memory as it was: nothing is allocated per call, whatever the size."""
    import torch
    run_pair(tr, (10_000, 10), seed=3)           # first use on this device, if the file runs alone
    a = torch.from_numpy(counts(tr.SCAN_STATIC_MAX_N, 5)).cuda()
    o = torch.empty(a.numel() + 1, dtype=torch.int32, device="cuda")
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    for n in (a.numel(), 77, 3_000_000):
        tr.tpc_scan_exclusive_static(a.data_ptr(), n, o.data_ptr())
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 == free0, (free0, free1)
