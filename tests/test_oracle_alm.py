"""Pins for oracle Part 2 (oracle/alm.py): exact line search against a brute-force scan, Lanczos
against a dense eigen-solver, and the full ALORA loop against closed-form optima (MaxCut K_n and
odd cycles, Lovasz theta) and the paper's Prop. 6 instance (the pass/fail test for rank
adaptation: without the growth step ALM never leaves the spurious point).  CPU only."""
import json
import os

import numpy as np
import pytest

from paper_2505_15775_b200 import inputs
from tests.test_oracle_pins import _graph_maxcut, prop6_instance

GOLD = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "paper_examples.json")))


@pytest.fixture(scope="module")
def Oracle(oracle_mod):
    return oracle_mod.Oracle


@pytest.fixture(scope="module")
def alm():
    from oracle import alm
    return alm


def test_counter_uniform(alm):
    """Start-vector generator [9] against literal values computed with exact Python integers
    (tests/golden/make_counter_uniform.py, which imports nothing from this repo) and against its statistics."""
    for c in GOLD["counter_uniform"]["cases"]:
        v = alm.counter_uniform(c["seed"], c["i"] + 1)
        assert v[c["i"]] == c["v"], c
    v = alm.counter_uniform(7, 100000)
    assert np.all(np.abs(v) < 1) and abs(v.mean()) < 0.01 and abs(v.var() - 1 / 3) < 0.01
    assert not np.array_equal(v[:100], alm.counter_uniform(8, 100))


def _dense_bfgs_inverse(S_list, Y_list, n):
    """Textbook BFGS inverse-Hessian recursion H <- (I - rho s y^T) H (I - rho y s^T) + rho s s^T applied to the
    pairs oldest first, from H_0 = (s^T y / y^T y) I of the NEWEST pair (Nocedal & Wright, eq. 6.17 / 7.20)."""
    s, y = S_list[-1], Y_list[-1]
    H = (s @ y) / (y @ y) * np.eye(n)
    for s, y in zip(S_list, Y_list):
        rho = 1.0 / (y @ s)
        V = np.eye(n) - rho * np.outer(y, s)
        H = V.T @ H @ V + rho * np.outer(s, s)
    return H


@pytest.mark.parametrize("npairs", [1, 2, 3, 5])
def test_lbfgs_direction_equals_dense_bfgs(alm, npairs):
    """The two-loop recursion [5] must give D = -H g with H the dense BFGS inverse Hessian built from the same
    pairs (a wrong sign of rho, a wrong loop order, or the scaling of the oldest pair all fail here)."""
    rng = np.random.default_rng(100 + npairs)
    n = 12
    A = rng.standard_normal((n, n)); A = A @ A.T + n * np.eye(n)      # pairs from a convex quadratic: s^T y > 0
    S_list = [rng.standard_normal(n) for _ in range(npairs)]
    Y_list = [A @ s for s in S_list]
    g = rng.standard_normal(n)
    D = alm.lbfgs_direction(g, S_list, Y_list)
    ref = -_dense_bfgs_inverse(S_list, Y_list, n) @ g
    assert np.linalg.norm(D - ref) <= 1e-12 * np.linalg.norm(ref)
    # matrix-shaped arguments (the loop hands over n x r arrays): same numbers
    D2 = alm.lbfgs_direction(g.reshape(4, 3), [s.reshape(4, 3) for s in S_list], [y.reshape(4, 3) for y in Y_list])
    np.testing.assert_allclose(D2.ravel(), D, rtol=1e-13, atol=1e-15)
    assert np.array_equal(alm.lbfgs_direction(g, [], []), -g)


def test_lbfgs_exact_steps_terminate_like_cg(alm):
    """On a strictly convex quadratic with exact steps and memory >= n, the L-BFGS iterates coincide with those
    of conjugate gradients (textbook: BFGS with exact line searches generates conjugate directions), so the
    gradient vanishes after at most n steps."""
    rng = np.random.default_rng(5)
    n = 10
    A = rng.standard_normal((n, n)); A = A @ A.T + np.eye(n)
    b = rng.standard_normal(n)
    x = np.zeros(n); g = A @ x - b
    xc = np.zeros(n); rc = b - A @ xc; pc = rc.copy()               # CG (Hestenes-Stiefel)
    S_list, Y_list = [], []
    for it in range(n):
        d = alm.lbfgs_direction(g, S_list, Y_list)
        alpha = -(g @ d) / (d @ A @ d)
        x_new = x + alpha * d; g_new = A @ x_new - b
        S_list.append(x_new - x); Y_list.append(g_new - g)
        x, g = x_new, g_new
        ac = (rc @ rc) / (pc @ A @ pc); xc = xc + ac * pc
        rn = rc - ac * (A @ pc); pc = rn + (rn @ rn) / (rc @ rc) * pc; rc = rn
        assert np.linalg.norm(x - xc) <= 1e-8 * (1 + np.linalg.norm(xc)), it
    assert np.linalg.norm(g) <= 1e-8 * np.linalg.norm(b)


def _sqrtf(expr):
    return float(eval(expr, {"sqrt": np.sqrt}))


def test_kkt_terms_hand_computed(alm, Oracle):
    """eq. 77 on the data of eq. 36, values worked out by hand in
    tests/golden/paper_examples.json["eq36_kkt"]; and exact zeros at the K_n primal-dual certificate."""
    from tests.helpers import problem_from_lists
    P = problem_from_lists(2, [], [[(0, 0, 1.0)], [(0, 1, 0.5)], [(0, 0, 1.0), (1, 1, 1.0)]], GOLD["eq36"]["b"])
    o = Oracle(P)
    for c in GOLD["eq36_kkt"]["cases"]:
        R = np.diag(np.sqrt(c["X_diag"])); y = np.array(c["y"])
        lam_min = np.linalg.eigvalsh(o.smatvec(y, np.eye(2)))[0]
        got = alm.kkt_at(o, R, y, lam_min)
        want = [_sqrtf(e) for e in c["kkt"]]
        np.testing.assert_allclose(got, want, rtol=1e-14, atol=1e-15)
    # the scalar form used inside the loop: l2 norms, the three "1 +" denominators, min{0, .}
    assert alm.kkt_terms(3.0, 1.0, -0.5, 3.0, 2.0, -1.0) == (1.5, 0.125, 0.75)
    assert alm.kkt_terms(0.0, 5.0, +0.7, 3.0, 2.0, 2.0) == (0.0, 0.0, 0.0)
    for n in (5, 9):
        Pk = _graph_maxcut(n, [(i, j) for i in range(n) for j in range(i + 1, n)])
        ok = Oracle(Pk)
        X = (n * np.eye(n) - np.ones((n, n))) / (n - 1)
        mu, Q = np.linalg.eigh(X)
        R = Q[:, 1:] * np.sqrt(mu[1:])
        ystar = np.full(n, -n / 4)
        lam_min = np.linalg.eigvalsh(ok.smatvec(ystar, np.eye(n)))[0]
        assert max(alm.kkt_at(ok, R, ystar, lam_min)) < 1e-13


def test_shrink_keeps_X_when_directions_are_null(alm, Oracle):
    """[13] R <- R Q_keep drops only null directions of R: X = RR^T, hence f, z = A(X) and ||G||_F, are unchanged
    to rounding, G(R Q) = G(R) Q, and the rank is the true rank; a full-rank R is left alone."""
    w = inputs.small(3)
    o = Oracle(w.problem)
    rng = np.random.default_rng(8)
    n, r1, r = w.problem.n, 4, 9
    Q0, _ = np.linalg.qr(rng.standard_normal((r, r)))
    R = np.hstack([rng.standard_normal((n, r1)) / np.sqrt(n), np.zeros((n, r - r1))]) @ Q0   # rank 4 inside 9 columns
    R2, dropped = alm.shrink_rank(R, 1e-8)
    assert dropped == r - r1 and R2.shape == (n, r1)
    np.testing.assert_allclose(R2 @ R2.T, R @ R.T, atol=1e-15)
    y, sg = w.y, w.sigma
    f1, f2 = o.f(y, sg, R), o.f(y, sg, R2)
    assert abs(f1 - f2) <= 1e-12 * (1 + abs(f1))
    np.testing.assert_allclose(o.A_op(R2), o.A_op(R), rtol=0, atol=1e-14 * (1 + np.abs(o.A_op(R)).max()))
    G1, G2 = o.grad(y, sg, R), o.grad(y, sg, R2)
    assert abs(np.linalg.norm(G1) - np.linalg.norm(G2)) <= 1e-12 * np.linalg.norm(G1)
    Qk = np.linalg.lstsq(R, R2, rcond=None)[0]                     # R2 = R Qk
    np.testing.assert_allclose(G1 @ Qk, G2, atol=1e-12 * np.abs(G1).max())
    R3, d3 = alm.shrink_rank(rng.standard_normal((50, 5)), 1e-8)
    assert d3 == 0 and R3.shape == (50, 5)
    # threshold is relative to the largest eigenvalue of R^T R: a direction at 1e-5 of the largest singular value
    # (mu ratio 1e-10) goes, one at 1e-3 (ratio 1e-6) stays, whatever the scale of R
    U, _ = np.linalg.qr(rng.standard_normal((50, 3)))
    R4, d4 = alm.shrink_rank(U * np.array([100.0, 0.1, 1e-3]), 1e-8)
    assert d4 == 1 and R4.shape == (50, 2)


def test_quartic_argmin_bruteforce(alm):
    rng = np.random.default_rng(3)
    for _ in range(200):
        p = rng.standard_normal(5)
        p[4] = abs(p[4]) + 1e-3
        p[1] = -abs(p[1])
        a, flag = alm.quartic_argmin(p)
        assert flag == 0 and a > 0
        grid = np.linspace(0, 2 * a + 5, 200001)[1:]
        phi = np.polyval(p[::-1], grid)
        assert np.polyval(p[::-1], a) <= phi.min() + 1e-9 * (1 + abs(phi.min()))
        assert abs(p[1] + a * (2 * p[2] + a * (3 * p[3] + 4 * p[4] * a))) < 1e-8 * (1 + np.abs(p).sum() * max(1, a) ** 3)
    assert alm.quartic_argmin([0, -2.0, 4.0, 0, 0]) == (0.25, 0)
    assert alm.quartic_argmin([0, -2.0, -1.0, 0, 0])[1] == 1


def test_lanczos_dense(alm, Oracle):
    w = inputs.small(0)
    o = Oracle(w.problem)
    lam, _ = o.lam(np.random.default_rng(1).standard_normal(w.problem.m), 1.0, w.R)
    S = o.smatvec(lam, np.eye(w.problem.n))
    ev, Q = np.linalg.eigh(S)
    theta, v, k, resid = alm.lanczos(lambda x: o.smatvec(lam, x), w.problem.n, 42, 300, 1e-8)
    assert abs(theta - ev[0]) < 1e-8 and k < 300
    assert np.linalg.norm(S @ v - theta * v) < 1e-6
    # breakdown: Prop. 6 operator has two distinct eigenvalues -> exact after 2 steps
    P, y, F, rho, eps, a = prop6_instance()
    o6 = Oracle(P)
    theta, v, k, resid = alm.lanczos(lambda x: o6.smatvec(y, x), P.n, 1, 50, 1e-12)
    assert k == 2 and abs(theta + eps) < 1e-14 and abs(abs(v[-1]) - 1) < 1e-12


@pytest.mark.parametrize("n", [9, 20])
def test_solve_Kn(alm, Oracle, n):
    P = _graph_maxcut(n, [(i, j) for i in range(n) for j in range(i + 1, n)])
    o = Oracle(P)
    R0 = inputs._unit_rows(np.random.default_rng(n), n, 4)
    res = alm.solve(o, R0, np.zeros(n), 1.0, alm.Params(eps=1e-7))
    assert res.converged
    assert abs(o.inner_C(res.R, res.R) + n * n / 4) < 1e-4
    assert np.abs(res.y + n / 4).max() < 1e-4


@pytest.mark.parametrize("n", [7, 51])
def test_solve_odd_cycle(alm, Oracle, n):
    P = _graph_maxcut(n, [(i, (i + 1) % n) for i in range(n)])
    o = Oracle(P)
    R0 = inputs._unit_rows(np.random.default_rng(n), n, 3)
    res = alm.solve(o, R0, np.zeros(n), 1.0, alm.Params(eps=1e-7))
    opt = -(n / 2) * (1 + np.cos(np.pi / n))
    assert res.converged and abs(o.inner_C(res.R, res.R) - opt) < 1e-5 * abs(opt)
    assert np.abs(res.y + 0.5 * (1 + np.cos(np.pi / n))).max() < 1e-4


def test_solve_from_rank_one_grows(alm, Oracle):
    """MaxCut on G(60,150) started from r0 = 1 must grow and reach the optimum found from r0 = 12."""
    rng = inputs._rng(77)
    lo, hi = inputs.gnm_edges(rng, 60, 150)
    P = inputs.maxcut_problem(60, lo, hi, np.ones(150))
    o = Oracle(P)
    a = alm.solve(o, inputs._unit_rows(rng, 60, 12), np.zeros(60), 1.0, alm.Params(eps=1e-7))
    b = alm.solve(o, inputs._unit_rows(rng, 60, 1), np.zeros(60), 1.0, alm.Params(eps=1e-7))
    assert a.converged and b.converged and any(r.grew for r in b.log)
    assert abs(o.inner_C(a.R, a.R) - o.inner_C(b.R, b.R)) < 1e-4


@pytest.mark.parametrize("name,n,edges,theta", [
    ("C5", 5, [(i, (i + 1) % 5) for i in range(5)], GOLD["theta"]["C5"]),
    ("C7", 7, [(i, (i + 1) % 7) for i in range(7)], 7 * np.cos(np.pi / 7) / (1 + np.cos(np.pi / 7))),
    ("K6", 6, [(i, j) for i in range(6) for j in range(i + 1, 6)], 1.0),
    ("empty6", 6, [], 6.0)])
def test_solve_theta(alm, Oracle, name, n, edges, theta):
    lo = np.array([e[0] for e in edges], np.int64); hi = np.array([e[1] for e in edges], np.int64)
    P = inputs.theta_problem(n, lo, hi)
    o = Oracle(P)
    R0 = np.random.default_rng(5).standard_normal((n, 3)) / np.sqrt(3 * n)
    res = alm.solve(o, R0, np.zeros(P.m), 1.0, alm.Params(eps=1e-7))
    assert res.converged, res.kkt
    assert abs(o.inner_C(res.R, res.R) + theta) < 2e-5 * theta


def test_prop6_escape(alm, Oracle):
    """Started at the spurious local minimiser F-hat with y = [0,..,0,2]: with the
    growth step ALORA reaches X* = a e_d e_d^T (objective eps*a, y* = [0,..,0,1]); with growth
    disabled it halts at F-hat forever (zero inner iterations, dual infeasible)."""
    P, y, F, rho, eps, a = prop6_instance()
    o = Oracle(P)
    fixed = dict(gamma=1.0, eps=1e-8)
    res = alm.solve(o, F, y, rho, alm.Params(**fixed))
    assert res.converged and res.log[0].grew == 1 and res.log[0].inner_iters == 0
    X = res.R @ res.R.T
    Xs = np.zeros((P.n, P.n)); Xs[-1, -1] = a
    assert np.abs(X - Xs).max() < 1e-5 and abs(o.inner_C(res.R, res.R) - eps * a) < 1e-6
    assert np.abs(res.y - np.r_[np.zeros(P.n - 1), 1.0]).max() < 1e-5
    stuck = alm.solve(o, F, y, rho, alm.Params(tau_neg=1e30, T_max=40, **fixed))
    assert not stuck.converged and all(r.inner_iters == 0 for r in stuck.log)
    assert abs(o.inner_C(stuck.R, stuck.R) - 2 * eps * a) < 1e-12 and stuck.kkt[1] > 1e-3


def test_config0_full_solve(alm, Oracle):
    """BASELINE.json config 0 to KKT <= 1e-6; first-order condition (5a) holds at
    the end: A(X) - b = (y_prev - y)/sigma by construction, and ||AX - b|| decreases overall."""
    w = inputs.full(0)
    o = Oracle(w.problem)
    res = alm.solve(o, w.R, w.y, w.sigma, alm.Params(eps=1e-6))
    assert res.converged and max(res.kkt) <= 1e-6
    assert res.log[-1].qnorm < 1e-3 * res.log[0].qnorm
    assert res.log[-1].r < 40 and any(r.shrank for r in res.log)
    # Barvinok-Pataki: final rank r(r+1)/2 <= m
    r = res.R.shape[1]
    assert r * (r + 1) // 2 <= w.problem.m


def test_thm1_bound_7b(alm, Oracle):
    """(7b) PAPER.md:250: ||A X_{y,rho} - b|| <= ||y - y*||/rho for an exact subproblem solution;
    K_9 with y* = -(9/4) 1, one outer iteration with a tight inner tolerance."""
    n = 9
    P = _graph_maxcut(n, [(i, j) for i in range(n) for j in range(i + 1, n)])
    o = Oracle(P)
    rng = np.random.default_rng(2)
    ystar = np.full(n, -n / 4)
    for rho in [0.5, 3.0]:
        y = ystar + 0.3 * rng.standard_normal(n)
        res = alm.solve(o, inputs._unit_rows(rng, n, n), y, rho,
                        alm.Params(T_max=1, tol0=1e-10, tol_min=1e-12, it_max=5000, tau_neg=1e30, gamma=1.0))
        q = o.A_op(res.R) - P.b
        assert np.linalg.norm(q) <= np.linalg.norm(y - ystar) / rho * (1 + 1e-6)
        # (8a) dual non-expansiveness: z = y - rho q is the updated dual
        assert np.linalg.norm(res.y - ystar) <= np.linalg.norm(y - ystar) * (1 + 1e-6)


def test_matrix_completion_nuclear_norm(alm, Oracle):
    """PAPER.md:997-1008 (section 6.2): with enough observations the SDP recovers M = U V^T exactly, and then
    its optimal value 1/2 tr X equals the nuclear norm of M (textbook: ||Y||_* = min 1/2 (tr W1 + tr W2)).
    Pins the general-class loop (single off-diagonal-entry constraints, C = I/2) against an SVD."""
    rng = np.random.default_rng(11)
    n1 = n2 = 20
    P, U, V = inputs.matrix_completion_problem(rng, n1, n2, 2, 300)   # 300 of 400 entries observed
    M = U @ V.T
    o = Oracle(P)
    R0 = rng.standard_normal((P.n, 4))
    res = alm.solve(o, R0, np.zeros(P.m), 1.0, alm.Params(eps=1e-7))
    assert res.converged
    X = res.R @ res.R.T
    Y = X[:n1, n1:]
    assert np.linalg.norm(Y - M) <= 1e-4 * np.linalg.norm(M)
    nuc = np.linalg.svd(M, compute_uv=False).sum()
    assert abs(o.inner_C(res.R, res.R) - nuc) <= 1e-5 * nuc


def test_lanczos_multi_rayleigh(alm, Oracle):
    """[29] several Ritz pairs of one run: orthonormal vectors whose Rayleigh quotients are the Ritz values
    (so U^T S U = diag(theta) whether or not they have converged); the converged ones match a dense solver."""
    w = inputs.small(0)
    o = Oracle(w.problem)
    lam, _ = o.lam(np.random.default_rng(1).standard_normal(w.problem.m), 1.0, w.R)
    S = o.smatvec(lam, np.eye(w.problem.n))
    theta, v, k, resid, (ths, U) = alm.lanczos(lambda x: o.smatvec(lam, x), w.problem.n, 42, 300, 1e-8, p_want=4)
    assert ths.shape == (4,) and U.shape == (w.problem.n, 4) and abs(ths[0] - theta) < 1e-12
    np.testing.assert_allclose(U.T @ U, np.eye(4), atol=1e-10)
    np.testing.assert_allclose(U.T @ S @ U, np.diag(ths), atol=1e-8)
    ev = np.linalg.eigvalsh(S)
    assert abs(ths[0] - ev[0]) < 1e-8 and np.all(ths >= ev[:4] - 1e-9)   # Ritz values interlace from above


def test_growth_sdp_model_and_optimality(alm, Oracle):
    """Alg. 1 line 7: g(S) = <U^T S(lambda) U, S> + sigma/2 ||A(U S U^T)||^2 is exactly
    L_rho(X + U S U^T, y) - L_rho(X, y); the computed S* is feasible, satisfies the KKT conditions of the
    small SDP (gradient psd, complementary to S*), beats random feasible points, and for p = 1 equals the
    closed form s* = -theta / (sigma ||A(vv^T)||^2) [10]."""
    rng = np.random.default_rng(5)
    w = inputs.small(3)                        # general class: dense-ish A(vv^T)
    P = w.problem
    o = Oracle(P)
    R, y, sigma = w.R, w.y, 0.7
    lam, _ = o.lam(y, sigma, R)
    n = P.n
    # three orthonormal directions with negative curvature: bottom Ritz vectors of S(lambda)
    _, _, _, _, (ths, U) = alm.lanczos(lambda x: o.smatvec(lam, x), n, 3, 60, 1e-10, p_want=3)
    assert np.all(ths < 0)
    pairs = [(a, c) for a in range(3) for c in range(a, 3)]
    cab = np.array([o.A_sym(U[:, [a]], U[:, [c]]) for a, c in pairs])
    H = cab @ cab.T
    M = U.T @ o.smatvec(lam, U)

    def g_model(S):
        v = sum((1.0 if a == c else 2.0) * S[a, c] * cab[i] for i, (a, c) in enumerate(pairs))
        return float(np.sum(M * S) + 0.5 * sigma * v @ v)

    f0 = o.f(y, sigma, R)
    for _ in range(3):
        A = rng.standard_normal((3, 3)) * 1e-3
        S = A @ A.T
        mu, Q = np.linalg.eigh(S)
        T = Q * np.sqrt(np.maximum(mu, 0))
        df = o.f(y, sigma, np.hstack([R, U @ T])) - f0
        assert abs(df - g_model(S)) <= 1e-9 * (abs(df) + abs(f0) * 1e-6 + 1e-12)
    S, gval = alm.growth_sdp(ths, H, sigma)
    assert np.linalg.eigvalsh(S)[0] >= -1e-12 and gval < 0
    assert abs(gval - g_model(S)) <= 1e-7 * abs(gval) + 1e-7 * np.abs(M - np.diag(ths)).max()
    # KKT of min g over the psd cone: G = dg/dS psd, <G, S> = 0
    v = sum((1.0 if a == c else 2.0) * S[a, c] * cab[i] for i, (a, c) in enumerate(pairs))
    G = np.diag(ths).astype(float)
    for i, (a, c) in enumerate(pairs):
        t = sigma * float(cab[i] @ v)
        G[a, c] += t
        if a != c:
            G[c, a] += t
    scale = np.abs(ths).max()
    assert np.linalg.eigvalsh(G)[0] >= -1e-5 * scale and abs(np.sum(G * S)) <= 1e-5 * scale * np.trace(S)
    for _ in range(2000):
        A = rng.standard_normal((3, 3)) * np.sqrt(np.trace(S)) * rng.random()
        assert g_model(A @ A.T) >= gval - 1e-9 * abs(gval)
    # p = 1 closed form
    S1, g1 = alm.growth_sdp(ths[:1], H[:1, :1], sigma)
    s_star = -ths[0] / (sigma * H[0, 0])
    assert abs(S1[0, 0] - s_star) <= 1e-12 * s_star and abs(g1 + 0.5 * ths[0] ** 2 / (sigma * H[0, 0])) <= 1e-12 * abs(g1)


def test_solve_pmax3_same_optimum(alm, Oracle):
    """p_max = 3 reaches the optimum that p_max = 1 reaches (MaxCut on G(60,150) from rank 1), growing by
    several columns in at least one outer iteration."""
    rng = np.random.default_rng(60)
    edges = set()
    while len(edges) < 150:
        i, j = sorted(int(x) for x in rng.integers(0, 60, 2))
        if i != j:
            edges.add((i, j))
    P = _graph_maxcut(60, sorted(edges))
    o = Oracle(P)
    R0 = inputs._unit_rows(np.random.default_rng(1), 60, 1)
    r1 = alm.solve(o, R0, np.zeros(60), 1.0, alm.Params(eps=1e-7, p_max=1))
    r3 = alm.solve(o, R0, np.zeros(60), 1.0, alm.Params(eps=1e-7, p_max=3))
    assert r1.converged and r3.converged and max(rec.grew for rec in r3.log) >= 2
    assert abs(o.inner_C(r1.R, r1.R) - o.inner_C(r3.R, r3.R)) <= 1e-5 * abs(o.inner_C(r1.R, r1.R))
