"""alora_rowdots_static -- the allocation-free entry point (scratch in a static __device__ array inside the library,
include/alora.h) -- against the existing alora_rowdots, which keeps the same partial sums in a cudaMalloc'ed workspace.
Both accumulate in fp64, in different orders; they must agree within the tolerances the parity tests use
(1e-10 on fp64 contexts, 2e-5 on fp32 ones).  Two calls in a row: the array is shared and keeps the last call's
contents, so the second call (a smaller shape, then a larger one) must not see the first one's partial rows or a stale
ticket.  Named test_zz_* so that pytest collects it last (the suite runs with pytest -x)."""
import numpy as np
import pytest

from paper_2505_15775_b200 import inputs

pytestmark = pytest.mark.gpu

TOL = {inputs.F64: 1e-10, inputs.F32: 2e-5}


@pytest.fixture(scope="module")
def torch():
    import torch
    assert torch.cuda.is_available(), "these tests need a CUDA device"
    return torch


@pytest.fixture(scope="module")
def binding():
    from paper_2505_15775_b200 import binding
    return binding


def close(got, ref, tol):
    # X.X is a sum of squares; X.Y cancels, so it is measured against |X| |Y| (what bounds its rounding error)
    return abs(got[0] - ref[0]) <= tol * abs(ref[0]) and abs(got[1] - ref[1]) <= tol * max(abs(ref[1]), ref[2])


@pytest.mark.parametrize("idx", [1, 0])   # small(1): fp32 context, small(0): fp64 context
def test_static_scratch_matches_workspace_path_twice_in_a_row(torch, binding, idx):
    w = inputs.small(idx)
    tol = TOL[w.dtype]
    dt = torch.float32 if w.dtype == inputs.F32 else torch.float64
    ctx = binding.Context(w.problem, w.dtype)
    g = torch.Generator(device="cuda").manual_seed(77 + idx)
    out = torch.full((2,), float("nan"), dtype=torch.float64, device="cuda")
    # shapes: several 16384-element chunks with a ragged tail and a padded leading dimension; then a SMALLER shape
    # (fewer blocks than the call before: stale partial rows beyond its grid must be ignored); then a larger contiguous one
    for (n_rows, r, ld) in ((9001, 10, 12), (37, 3, 3), (200003, 16, 16), (1, 1, 5)):
        X = torch.randn(n_rows, ld, generator=g, dtype=dt, device="cuda")
        Y = torch.randn(n_rows, ld, generator=g, dtype=dt, device="cuda")
        ref = ctx.rowdots(X, Y, n_rows, r, ld)                         # existing path (allocating workspace)
        bound = float(torch.linalg.norm(X[:, :r].double()) * torch.linalg.norm(Y[:, :r].double()))
        for call in range(2):                                            # two calls in a row on the shared array
            out.fill_(float("nan"))
            ctx.rowdots_static(X, Y, n_rows, r, ld, out)
            got = out.cpu().numpy()
            assert close(got, (ref[0], ref[1], bound), tol), (n_rows, r, ld, call, got, ref)
        # and against a direct fp64 sum, so that a defect common to both paths cannot hide
        Xd, Yd = X[:, :r].double(), Y[:, :r].double()
        direct = (float((Xd * Xd).sum()), float((Xd * Yd).sum()), bound)
        assert close(got, direct, tol), (n_rows, r, ld, got, direct)
    # empty input: zeros, no launch
    out.fill_(float("nan"))
    ctx.rowdots_static(X, Y, 0, 1, 5, out)
    assert out.cpu().tolist() == [0.0, 0.0]
    ctx.close()


def test_static_scratch_rejects_shapes_beyond_its_maximum(torch, binding):
    w = inputs.small(1)
    ctx = binding.Context(w.problem, w.dtype)
    X = torch.zeros(8, 4, dtype=torch.float32, device="cuda")
    out = torch.full((2,), 5.0, dtype=torch.float64, device="cuda")
    lim = binding.ROWDOTS_STATIC_MAX_ELEMS
    for (n_rows, r) in ((lim // 4 + 1, 4), (lim + 1, 1), (2 ** 62, 64)):   # validated before anything is read
        with pytest.raises(binding.AloraError) as e:
            ctx.rowdots_static(X, X, n_rows, r, r, out)
        assert e.value.status == binding.EINVAL
        assert "maximum" in str(e.value) and str(lim) in str(e.value), str(e.value)
    torch.cuda.synchronize()
    assert out.cpu().tolist() == [5.0, 5.0]                               # a rejected call writes nothing
    # exactly at the limit the shape is accepted (4096 blocks, every partial row of the array in use)
    n_rows, r = lim // 16, 16
    Xb = torch.full((n_rows, r), 0.5, dtype=torch.float32, device="cuda")
    Yb = torch.full((n_rows, r), -2.0, dtype=torch.float32, device="cuda")
    ctx.rowdots_static(Xb, Yb, n_rows, r, r, out)
    assert out.cpu().tolist() == [0.25 * lim, -1.0 * lim]                 # exact in fp64
    ctx.close()
