"""tina_sum_static: the entry point that allocates no device memory (partial sums in a file-scope `static __device__`
array, include/tina.h).  Kept in a file pytest collects LAST: the run uses -x, so a failure here hides
nothing.  Passes alone in a fresh process (first use looks the scratch address up) and after the other tests."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def tina():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_2408_16551_b200 as t
    t.lib()  # raises if libtina.so is missing -- no fallback
    return t


def test_sum_static_matches_sum_two_calls_in_a_row(tina, oracle):
    """Two calls in a row through the shared static scratch, the second with fewer rows and fewer partials per row
    than the first (stale partials of call 1 stay in the array): each must equal tina_sum on the same input, within
    the tolerance of test_arith_sum (|got - ref| <= 1e-6 sum|x| + one float32 rounding); in fact bit-identical,
    since both use the same decomposition.  Also against the float64 oracle."""
    import torch
    rng = np.random.default_rng(4242)
    shapes = [(37, 4096 * 29 + 13), (5, 4096 * 3 + 1)]
    xs = [torch.from_numpy((rng.standard_normal(s) + 0.25).astype(np.float32)).cuda() for s in shapes]
    outs = [torch.full((s[0],), float("nan"), device="cuda") for s in shapes]
    refs = [tina.summation(x) for x in xs]                 # existing path (cudaMallocAsync temporary)
    torch.cuda.synchronize()
    before = torch.cuda.memory_allocated()
    launches = tina.launch_count()
    for x, o in zip(xs, outs):                             # back to back on one stream, no sync in between
        tina.summation_static(x, o)
    torch.cuda.synchronize()
    assert tina.launch_count() - launches == 4
    assert tina.last_kernel() == "sum_kernel<static scratch>"
    assert torch.cuda.memory_allocated() == before
    for x, o, r in zip(xs, outs, refs):
        xh = x.cpu().numpy()
        got, ref = o.cpu().numpy().astype(np.float64), r.cpu().numpy().astype(np.float64)
        tol = 1e-6 * np.abs(xh).sum(axis=1, dtype=np.float64) + 6e-8 * np.abs(ref) + 1e-30
        assert np.all(np.abs(got - ref) <= tol)
        assert np.array_equal(o.cpu().numpy(), r.cpu().numpy())
        assert np.all(np.abs(got - oracle.summation(xh)) <= tol)


@pytest.mark.parametrize("rows,n", [(1, 0), (1, 1), (3, 1000), (2, 1 << 22), (4096, 64), (1500, 9000)])
def test_sum_static_shapes(tina, rows, n):
    """Single block per row, many blocks per row, the row limit itself; 1-D input."""
    import torch
    rng = np.random.default_rng(77 + rows)
    x = torch.from_numpy(rng.standard_normal((rows, n)).astype(np.float32)).cuda()
    out = torch.full((rows,), float("nan"), device="cuda")
    tina.summation_static(x, out)
    ref = tina.summation(x)
    torch.cuda.synchronize()
    assert np.array_equal(out.cpu().numpy(), ref.cpu().numpy())
    if n:
        one = torch.full((1,), float("nan"), device="cuda")
        tina.summation_static(x[0], one)
        ref1 = tina.summation(x[0])                        # a one-row call splits the row over more blocks
        torch.cuda.synchronize()
        assert float(one[0]) == float(ref1)


def test_sum_static_rejects_beyond_the_limit(tina):
    import torch
    L = tina.lib()
    x = torch.zeros(4097 * 4, device="cuda")
    out = torch.zeros(4097, device="cuda")
    assert L.tina_sum_static(x.data_ptr(), 4097, 4, out.data_ptr(), None) == 3          # UNSUPPORTED
    assert b"4096" in L.tina_last_error()
    assert L.tina_sum_static(x.data_ptr(), -1, 4, out.data_ptr(), None) == 2            # BAD_SHAPE
    assert L.tina_sum_static(None, 2, 4, out.data_ptr(), None) == 1                     # NULL_POINTER
    assert L.tina_sum_static(x.data_ptr(), 0, 4, None, None) == 0                       # nothing to do
    with pytest.raises(tina.TinaError):
        tina.summation_static(x.view(4097, 4), out)
