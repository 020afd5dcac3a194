"""lrp_topk_static (include/lrp.h): the allocation-free top-k entry point with its scratch in a device array built into the
library, against the existing workspace path (lrp_leverage_select on the same scores), bit for bit, on two calls in a row
of different shape -- the second call finds the first call's candidates in the shared scratch and must not consume them.
Collected last on purpose (the file name): a failure here hides no other test under `pytest -x`."""
import ctypes as C

import numpy as np
import pytest

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def ctx():
    from paper_2607_06021_b200 import build, lrp
    build.build()
    c = lrp.Context(0)
    yield c
    c.close()


def _existing_path(ctx, n, num, seed):
    """scores = a(i)^2 of a one-column block used as Q (assume_orthonormal = 1) -> (scores, indices) of the workspace path;
    a few exact ties (repeated values) exercise the index-ascending tie rule."""
    import torch
    rng = np.random.default_rng(seed)
    a = rng.standard_normal(n)
    a[rng.integers(0, n, 64)] = a[rng.integers(0, n)]             # ties
    a[rng.integers(0, n, 8)] = 7.5                                 # ties among the largest
    A = torch.from_numpy(a.reshape(1, n)).cuda()
    idx, scores = ctx.leverage_select(A, num, assume_orthonormal=True)
    return scores, idx.cpu().numpy().copy()


def test_topk_static_matches_workspace_path_twice_in_a_row(ctx):
    import torch
    from paper_2607_06021_b200 import lrp
    # three levels, ragged last chunk, then a smaller call with fewer candidates per level, then a one-chunk call
    shapes = [(1_000_003, 200, 11), (300_001, 72, 12), (5000, 256, 13), (lrp.TOPK_STATIC_MAX_N, 256, 14)]
    refs = [_existing_path(ctx, n, num, seed) for n, num, seed in shapes]
    outs = [torch.full((num,), -7, dtype=torch.int32, device="cuda") for _, num, _ in shapes]
    torch.cuda.synchronize()
    lrp.topk_static(refs[0][0], shapes[0][1], outs[0])            # first call on this device: symbol address looked up here
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    for (n, num, _), (scores, _), out in zip(shapes[1:], refs[1:], outs[1:]):   # back to back on one stream, no sync between
        lrp.topk_static(scores, num, out)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0                   # nothing was allocated or freed on the device
    for (n, num, _), (scores, ref), out in zip(shapes, refs, outs):
        got = out.cpu().numpy()
        assert np.array_equal(got, ref), (n, num)
        # and against the definition: (score descending, index ascending)
        s = scores.cpu().numpy()
        order = np.lexsort((np.arange(n), -s))[:num]
        assert np.array_equal(got, order.astype(np.int32))
    # the same first call again (the scratch now holds the last call's candidates)
    again = torch.empty(shapes[0][1], dtype=torch.int32, device="cuda")
    lrp.topk_static(refs[0][0], shapes[0][1], again)
    assert np.array_equal(again.cpu().numpy(), refs[0][1])


def test_topk_static_on_a_side_stream_and_limits(ctx):
    import torch
    from paper_2607_06021_b200 import lrp
    scores, ref = _existing_path(ctx, 70_001, 33, 21)
    st = torch.cuda.Stream()
    out = torch.empty(33, dtype=torch.int32, device="cuda")
    st.wait_stream(torch.cuda.current_stream())
    lrp.topk_static(scores, 33, out, stream=st)
    st.synchronize()
    assert np.array_equal(out.cpu().numpy(), ref)
    assert lrp.topk_static(scores, 0, out).numel() == 0           # num_select = 0: nothing to do
    lib = lrp.load_library()
    big = torch.zeros(16, dtype=torch.float64, device="cuda")      # the limits are checked before any memory is touched
    o = torch.empty(512, dtype=torch.int32, device="cuda")
    assert lib.lrp_topk_static(None, lrp.TOPK_STATIC_MAX_N + 1, big.data_ptr(), 4, o.data_ptr()) == lrp.LRP_ERR_STATIC_LIMIT
    assert lib.lrp_topk_static(None, 1 << 20, big.data_ptr(), lrp.TOPK_STATIC_MAX_NUM + 1, o.data_ptr()) == lrp.LRP_ERR_STATIC_LIMIT
    assert lib.lrp_topk_static(None, 16, big.data_ptr(), 17, o.data_ptr()) == lrp.LRP_ERR_BADARG
    assert lib.lrp_topk_static(None, 16, None, 4, o.data_ptr()) == lrp.LRP_ERR_BADARG
    assert lib.lrp_topk_static(None, 16, big.data_ptr() + 4, 4, o.data_ptr()) == lrp.LRP_ERR_BADARG
    with pytest.raises(lrp.LrpError, match="fixed capacity"):
        lrp.topk_static(torch.zeros(1 << 20, dtype=torch.float64, device="cuda"), 300, o)
