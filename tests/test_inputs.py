"""Seeded input generators (paper_2505_15775_b200/inputs.py): determinism, the structure each recipe promises
 and the storage convention (sym-upper COO).  CPU only, small sizes."""
import numpy as np
import pytest

from paper_2505_15775_b200 import inputs


@pytest.mark.parametrize("idx", list(range(8)))
def test_small_configs_are_deterministic_and_well_formed(idx):
    a, b = inputs.small(idx), inputs.small(idx)
    P, Q = a.problem, b.problem
    for f in ("C_row", "C_col", "C_val", "A_ptr", "A_row", "A_col", "A_val", "b"):
        np.testing.assert_array_equal(getattr(P, f), getattr(Q, f))
    np.testing.assert_array_equal(a.R, b.R)
    np.testing.assert_array_equal(a.y, b.y)
    assert np.all(P.C_row <= P.C_col) and np.all(P.A_row <= P.A_col)          # sym-upper storage
    assert P.A_ptr[0] == 0 and P.A_ptr[-1] == P.nnzA and np.all(np.diff(P.A_ptr) >= 0)
    assert P.C_col.max(initial=0) < P.n and P.A_col.max(initial=0) < P.n
    assert a.R.shape == (P.n, a.r) and a.D.shape == a.R.shape and a.V.shape == (P.n,) and a.y.shape == (P.m,)
    if a.dtype == inputs.F32:   # fp32 workloads hand out fp32-representable values
        for x in (a.R, a.D, a.V, P.C_val, P.A_val):
            np.testing.assert_array_equal(x, x.astype(np.float32).astype(float))


def test_maxcut_cost_is_minus_quarter_laplacian():
    """C = -L/4 with L_ii = sum_k w_ik, L_ij = -w_ij; diagonal constraints X_ii = 1."""
    rng = np.random.default_rng(0)
    lo, hi = inputs.gnm_edges(rng, 30, 60)
    w = rng.choice([-1.0, 1.0], size=60)
    P = inputs.maxcut_problem(30, lo, hi, w)
    L = np.zeros((30, 30))
    for i, j, wv in zip(lo, hi, w):
        L[i, j] -= wv; L[j, i] -= wv; L[i, i] += wv; L[j, j] += wv
    Cd = np.zeros((30, 30))
    for i, j, v in zip(P.C_row, P.C_col, P.C_val):
        Cd[i, j] += v
        if i != j:
            Cd[j, i] += v
    np.testing.assert_allclose(Cd, -L / 4, atol=1e-15)
    assert P.m == 30 and np.all(P.A_row == np.arange(30)) and np.all(P.A_col == np.arange(30)) and np.all(P.b == 1)


def test_graph_shapes():
    lo, hi = inputs.torus_edges(7)
    assert lo.shape[0] == 2 * 49 and len(set(zip(lo.tolist(), hi.tolist()))) == 2 * 49
    lo, hi = inputs.tri_torus_edges(7)
    deg = np.bincount(np.concatenate([lo, hi]), minlength=49)
    assert lo.shape[0] == 3 * 49 and np.all(deg == 6)
    lo, hi = inputs.ring_matching_edges(np.random.default_rng(1), 1000)
    deg = np.bincount(np.concatenate([lo, hi]), minlength=1000)
    assert lo.shape[0] == 2000 and np.all(deg == 4)        # ring (2) + two perfect matchings (1 + 1)
    lo, hi = inputs.rmat_edges(np.random.default_rng(2), 10, 8)
    deg = np.bincount(np.concatenate([lo, hi]), minlength=1024)
    assert lo.shape[0] == 8 * 1024 and deg.max() > 20 * np.median(deg[deg > 0])   # heavy tail


def test_matrix_completion_recipe():
    """M = U V^T, m distinct observed entries, constraint X[i, n1+j] = M_ij stored (i, n1+j, 1/2),
    C = I/2, m = ceil(r* log n r* (n - r*))."""
    rng = np.random.default_rng(3)
    P, U, V = inputs.matrix_completion_problem(rng, 12, 9, 2, 50)
    assert P.n == 21 and P.m == 50 and np.all(np.diff(P.A_ptr) == 1) and np.all(P.A_val == 0.5)
    assert np.all(P.A_row < 12) and np.all(P.A_col >= 12)
    assert len(set(zip(P.A_row.tolist(), P.A_col.tolist()))) == 50          # without replacement
    np.testing.assert_allclose(P.b, (U @ V.T)[P.A_row, P.A_col - 12])
    assert np.all(P.C_row == P.C_col) and np.all(P.C_val == 0.5) and P.nnzC == 21
    assert inputs.mc_observations(10000, 3) == int(np.ceil(3 * np.log(10000) * 3 * 9997))


def test_theta_and_planted_rhs(oracle_mod):
    P = inputs.theta_problem(5, np.array([0, 1, 2, 3, 0]), np.array([1, 2, 3, 4, 4]))
    assert P.m == 6 and P.A_ptr[1] == 5 and P.b[0] == 1 and np.all(P.b[1:] == 0) and P.pC == 1
    w = inputs.small(3)                      # b = A(R0 R0^T) for the planted R0: checked against the oracle's A
    o = oracle_mod.Oracle(w.problem)
    rng = np.random.default_rng(4)
    R0 = rng.standard_normal((w.problem.n, 3))
    b = inputs.planted_rhs(w.problem.A_ptr, w.problem.A_row, w.problem.A_col, w.problem.A_val, R0)
    np.testing.assert_allclose(b, o.A_op(R0), rtol=1e-12, atol=1e-12)
