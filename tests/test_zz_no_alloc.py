"""mlp_row_offsets_static: the allocation-free entry point (scratch in a static __device__ array) against the existing
scan path of the neighbour build (mlp_debug_row_offsets = the kernels mlp_compute launches, with a cudaMalloc'ed block
buffer).  Integer work: the bar is bit-exact.  Collected last on purpose (file name), so that under `pytest -x` a failure
here cannot hide another test; it must pass alone in a fresh process and after every other test.
"""
import numpy as np
import pytest

import paper_2506_04055_b200 as P

pytestmark = pytest.mark.gpu


def _counts(n, seed):
    # row lengths of a padded CSR neighbour list: multiples of 8, a few empty rows, a few long ones
    rng = np.random.default_rng(seed)
    c = 8 * rng.integers(0, 12, size=n)
    c[rng.random(n) < 0.02] = 0
    c[rng.random(n) < 0.001] = 8 * 40
    return c.astype(np.int32)


def test_static_row_offsets_match_the_existing_path_twice_in_a_row():
    import torch
    dev = torch.device("cuda:0")
    # calls in a row on the one shared array: 63 blocks + a ragged tail, then a SMALLER input that must not see what the
    # first left behind, then 1,221 blocks (more than one 1,024-wide pass of the top-level scan), then the degenerate sizes
    for n, seed in ((257_123, 1), (4_097, 2), (5_000_001, 3), (0, 4), (1, 5)):
        c = _counts(n, seed)
        d_c = torch.from_numpy(c).to(dev)
        off_ref, tot_ref = P.row_offsets(d_c, static=False)
        off_new, tot_new = P.row_offsets(d_c, static=True)
        torch.cuda.synchronize()
        expect = np.concatenate([[0], np.cumsum(c, dtype=np.int64)])
        assert int(tot_ref.item()) == int(expect[-1])
        assert int(tot_new.item()) == int(tot_ref.item()), n
        assert torch.equal(off_new, off_ref), n                       # the two CUDA paths agree bit for bit
        assert np.array_equal(off_new.cpu().numpy().astype(np.int64), expect), n   # and both are the plain definition


def test_static_row_offsets_allocate_nothing_and_accept_a_null_total():
    import torch
    dev = torch.device("cuda:0")
    n = 100_000
    c = _counts(n, 7)
    d_c = torch.from_numpy(c).to(dev)
    off = torch.full((n + 1,), -1, dtype=torch.int32, device=dev)
    tot = torch.zeros(1, dtype=torch.int64, device=dev)
    P.row_offsets_into(d_c, off, tot, static=True)                    # first use on this device: takes the symbol address
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info(dev)
    for _ in range(2):
        off.fill_(-1)
        P.row_offsets_into(d_c, off, None, static=True)               # total = NULL
        torch.cuda.synchronize()
        assert np.array_equal(off.cpu().numpy().astype(np.int64), np.concatenate([[0], np.cumsum(c, dtype=np.int64)]))
    free1, _ = torch.cuda.mem_get_info(dev)
    assert free1 == free0                                             # the driver handed out no device memory


def test_static_row_offsets_under_stream_capture():
    # the use case: a region where cudaMalloc is illegal.  Capture two calls into a CUDA graph and replay it.
    import torch
    dev = torch.device("cuda:0")
    n = 70_000
    c = _counts(n, 9)
    d_c = torch.from_numpy(c).to(dev)
    off = torch.zeros(n + 1, dtype=torch.int32, device=dev)
    tot = torch.zeros(1, dtype=torch.int64, device=dev)
    P.row_offsets_into(d_c, off, tot, static=True)                    # set-up outside the capture
    torch.cuda.synchronize()
    g = torch.cuda.CUDAGraph()
    s = torch.cuda.Stream(dev)
    with torch.cuda.stream(s):
        with torch.cuda.graph(g, stream=s):
            P.row_offsets_into(d_c, off, tot, static=True, stream=s.cuda_stream)
    off.zero_(); tot.zero_()
    d_c.copy_(torch.from_numpy(_counts(n, 10)).to(dev))               # new counts, same buffers
    g.replay()
    torch.cuda.synchronize()
    expect = np.concatenate([[0], np.cumsum(_counts(n, 10), dtype=np.int64)])
    assert int(tot.item()) == int(expect[-1])
    assert np.array_equal(off.cpu().numpy().astype(np.int64), expect)


def test_static_row_offsets_reject_sizes_beyond_the_static_scratch():
    import torch
    dev = torch.device("cuda:0")
    d_c = torch.zeros(8, dtype=torch.int32, device=dev)
    off = torch.zeros(9, dtype=torch.int32, device=dev)
    with pytest.raises(P.MLPError) as e:
        P.row_offsets_into(d_c, off, None, static=True, n=P.ROW_OFFSETS_STATIC_MAX + 1)
    assert e.value.code == 1                                          # MLP_ERR_ARG; nothing was launched
    with pytest.raises(P.MLPError):
        P.row_offsets_into(d_c, off, None, static=True, n=-1)
    torch.cuda.synchronize()
    assert int(off.abs().sum().item()) == 0
