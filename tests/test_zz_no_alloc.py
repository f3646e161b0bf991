"""oo_sort_queries_static: the Morton order for callers that cannot allocate device memory (an application past its
start-up phase with a frozen memory budget, a plug-in whose host owns the device heap, a real-time thread that cannot
afford cudaMalloc's device-wide synchronisation).  Its scratch is an array inside the library image instead of
oo_reserve's cudaMalloc, so this file checks that it returns exactly what the existing path (oo_reserve +
oo_sort_queries) returns — integer work, so the bar is bit-exact, as in test_morton_sort_and_permuted_query — and that
calls made one after the other do not see each other's leftovers in the shared array.

The file name sorts after every other test file on purpose: pytest -x stops at the first failure, and this test of an
add-on must never hide a failure of the hot path's own tests.  It makes no assumption on what ran before it in the
process (the library may or may not be loaded, other contexts may or may not exist)."""
import numpy as np
import pytest

import gen
from oracle import oo_oracle as O

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

GUARD = 64
SENTINEL = -17


def _positions(seed, n):
    # a cloud reaching past the unit cube on every side (keys clamp), as in the existing sort test
    return torch.from_numpy((gen.u01(seed, 1, 3 * n).reshape(-1, 3) * 1.2 - 0.1).astype(np.float32)).cuda()


def _static_sort(P, x):
    """Call the no-allocation entry point into a caller-owned output with guard rows behind it."""
    n = int(x.shape[0])
    out = torch.full((n + GUARD,), SENTINEL, dtype=torch.int32, device=x.device)
    got = P.oo_sort_queries_static(x, perm_out=out)
    assert got.data_ptr() == out.data_ptr()
    return out


def test_static_scratch_sort_equals_the_reserved_scratch_sort_on_consecutive_calls():
    import paper_2606_08469_b200 as P
    ctx = P.OctaOctree(0)
    # sizes: several 4096-key tiles with a ragged tail; then a LARGER batch, then a much smaller one, so that the second and
    # third call find the first one's keys, indices and histogram rows in the shared array, both inside and beyond their own n
    sizes = (70001, 300007, 4097, 1)
    ctx.oo_reserve(max(sizes))
    xs = [_positions(11 + k, n) for k, n in enumerate(sizes)]
    # all static calls back to back on one stream, nothing in between: this is the "two calls in a row" case
    outs = [_static_sort(P, x) for x in xs]
    torch.cuda.synchronize()
    for x, out in zip(xs, outs):
        n = int(x.shape[0])
        ref = ctx.oo_sort_queries(x)
        torch.cuda.synchronize()
        got = out.cpu().numpy()
        assert np.array_equal(got[:n], ref.cpu().numpy()), "static-scratch permutation differs from oo_sort_queries at n = %d" % n
        assert np.all(got[n:] == SENTINEL), "wrote past perm_out[n)"
        # and both are the unique stable Morton order the oracle defines
        assert np.array_equal(got[:n].astype(np.int64), O.morton_order(x.cpu().numpy()))
    # the same input again gives the same bytes (nothing of the calls in between survives in the result)
    again = _static_sort(P, xs[0])
    torch.cuda.synchronize()
    assert torch.equal(again, outs[0])
    ctx.close()


def test_static_scratch_sort_at_its_maximum_and_beyond():
    import paper_2606_08469_b200 as P
    nmax = P.SORT_STATIC_MAX_QUERIES
    assert nmax == 1 << 20
    x = _positions(5, nmax + 1)
    # n = 0: the set-up call; touches neither pointer
    P.oo_sort_queries_static(x[:0])
    # one more than the maximum: refused with a message that names the limit, nothing launched, output untouched
    out = torch.full((nmax + 1,), SENTINEL, dtype=torch.int32, device="cuda")
    with pytest.raises(P.OOError) as ei:
        P.oo_sort_queries_static(x, perm_out=out)
    assert ei.value.status == 3 and "OO_SORT_STATIC_MAX_QUERIES" in str(ei.value) and str(nmax) in str(ei.value)
    torch.cuda.synchronize()
    assert bool((out == SENTINEL).all())
    # exactly the maximum (the 1024 x 1024 frame): equal to the existing path
    xm = x[:nmax].contiguous()
    got = _static_sort(P, xm)
    ctx = P.OctaOctree(0)
    ctx.oo_reserve(nmax)
    ref = ctx.oo_sort_queries(xm)
    torch.cuda.synchronize()
    assert torch.equal(got[:nmax], ref) and bool((got[nmax:] == SENTINEL).all())
    # a refused call leaves nothing pending: the next one works
    again = _static_sort(P, xm)
    torch.cuda.synchronize()
    assert torch.equal(again, got)
    ctx.close()
