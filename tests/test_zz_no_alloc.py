"""reann_row_ptr_noalloc (include/reann.h): the scan of per-atom neighbour counts into CSR row pointers with its
workspace in a file-scope device array, for callers that cannot call cudaMalloc. Checked against the existing path:
the row pointers the handle's neighbour build produced (same kernels, workspace from cudaMalloc) -- integer work, so
the gate is bit-exact. Collected last (file name) so that a failure here cannot hide another test under `pytest -x`."""
import numpy as np
import pytest

import gen

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def R():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import __graft_entry__ as ge
    ge.build()
    import paper_2505_06711_b200 as R
    return R


def _existing_path_row_ptr(R, k):
    """row_ptr of the handle's neighbour build (the existing path) on BASELINE config k."""
    cfg = gen.make_config(k)
    m = R.Reann.from_config(cfg)
    m.build_neighbors(cfg["pos"], cfg["box"])
    row_ptr, _, _ = m.neighbors()
    m.close()
    return row_ptr


def test_no_alloc_row_ptr_matches_existing_path_twice_in_a_row(R):
    import torch
    dev = torch.device("cuda:0")
    # two calls in a row, the larger problem FIRST: the second call finds the first one's block totals and offsets
    # in the shared scratch and must not be disturbed by them
    refs = [_existing_path_row_ptr(R, 2), _existing_path_row_ptr(R, 1)]   # 3072 atoms (2 scan blocks), 96 atoms
    assert len(refs[0]) - 1 > 2048 > len(refs[1]) - 1
    counts = [torch.from_numpy(np.diff(r).astype(np.int32)).to(dev) for r in refs]
    outs = [torch.full((len(r),), -7, dtype=torch.int64, device=dev) for r in refs]
    torch.cuda.synchronize()
    stream = torch.cuda.current_stream().cuda_stream
    free0 = torch.cuda.mem_get_info()[0]
    for c, o in zip(counts, outs):                     # back to back on one stream, no sync in between
        R.reann_row_ptr_noalloc(c, c.numel(), o, stream)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0       # the device's free memory did not move
    for r, o in zip(refs, outs):
        assert np.array_equal(o.cpu().numpy(), r)      # bit-exact against the existing path
    # and once more in the other order, same buffers
    for c, o in zip(counts[::-1], outs[::-1]):
        o.fill_(-7)
        R.reann_row_ptr_noalloc(c, c.numel(), o, stream)
    torch.cuda.synchronize()
    for r, o in zip(refs, outs):
        assert np.array_equal(o.cpu().numpy(), r)


def test_no_alloc_row_ptr_three_levels_limit_and_errors(R):
    import torch
    dev = torch.device("cuda:0")
    rng = np.random.default_rng(11)
    stream = torch.cuda.current_stream().cuda_stream
    # the maximum size (three scan levels, sums beyond 2^31), then sizes around the block boundaries, then the
    # degenerate ones -- each call after a larger one
    for n in (R.REANN_NOALLOC_MAX_ROWS, 2048 * 2048 + 5, 2049, 2048, 2047, 1, 0):
        c_np = rng.integers(0, 400, size=n, dtype=np.int32)
        c = torch.from_numpy(c_np).to(dev)
        o = torch.full((n + 1,), -1, dtype=torch.int64, device=dev)
        R.reann_row_ptr_noalloc(c if n else None, n, o, stream)
        torch.cuda.synchronize()
        want = np.zeros(n + 1, dtype=np.int64)
        np.cumsum(c_np, dtype=np.int64, out=want[1:])
        assert np.array_equal(o.cpu().numpy(), want), n
        if n == R.REANN_NOALLOC_MAX_ROWS:
            assert want[-1] > 2 ** 31
    # beyond the limit: a clear error, nothing written
    o = torch.full((4,), -1, dtype=torch.int64, device=dev)
    with pytest.raises(R.ReannError) as ei:
        R.reann_row_ptr_noalloc(o, R.REANN_NOALLOC_MAX_ROWS + 1, o, stream)
    assert ei.value.code == R.REANN_ERR_UNSUPPORTED and "REANN_NOALLOC_MAX_ROWS" in str(ei.value)
    with pytest.raises(R.ReannError) as ei:
        R.reann_row_ptr_noalloc(None, 3, o, stream)
    assert ei.value.code == R.REANN_ERR_ARG
    torch.cuda.synchronize()
    assert (o.cpu().numpy() == -1).all()
