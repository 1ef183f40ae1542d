"""Pins for oracle Part 1 (oracle/alora_oracle.c) against what the paper and mathematics fix:
dense X = RR^T brute force, finite differences, the exact-quartic identity, the paper's worked
examples (values in tests/golden/paper_examples.json, each with its PAPER.md citation) and
special cases that reduce to a textbook formula.  CPU only."""
import json
import os

import numpy as np
import pytest

from paper_2505_15775_b200 import inputs
from tests.helpers import dense_matrices, problem_from_lists, random_problem

GOLD = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "paper_examples.json")))


@pytest.fixture(scope="module")
def Oracle(oracle_mod):
    return oracle_mod.Oracle


@pytest.mark.parametrize("seed,n,m,r,pC", [(0, 7, 5, 3, 0), (1, 33, 40, 4, 2), (2, 64, 100, 6, 1), (3, 12, 1, 12, 0)])
def test_dense_bruteforce(Oracle, seed, n, m, r, pC):
    """z, f, grad, S(mu)v, <C,XY^T>, ||C||_F against dense matrices (n <= 64)."""
    rng = np.random.default_rng(seed)
    P = random_problem(rng, n, m, pC=pC)
    o = Oracle(P)
    Cd, Ad = dense_matrices(P)
    R, D = rng.standard_normal((n, r)), rng.standard_normal((n, r))
    y, sigma = rng.standard_normal(m), 0.7
    X = R @ R.T
    z = np.array([np.sum(Ai * X) for Ai in Ad])
    np.testing.assert_allclose(o.A_op(R), z, rtol=1e-12, atol=1e-12)
    q = z - P.b
    f = np.sum(Cd * X) - y @ q + 0.5 * sigma * q @ q
    assert abs(o.f(y, sigma, R) - f) <= 1e-12 * (1 + abs(f))
    lam = y - sigma * q
    S = Cd - sum(l * Ai for l, Ai in zip(lam, Ad))
    np.testing.assert_allclose(o.grad(y, sigma, R), 2 * S @ R, rtol=1e-11, atol=1e-11)
    mu = rng.standard_normal(m)
    Smu = Cd - sum(l * Ai for l, Ai in zip(mu, Ad))
    V = rng.standard_normal((n, 3))
    np.testing.assert_allclose(o.smatvec(mu, V), Smu @ V, rtol=1e-11, atol=1e-11)
    np.testing.assert_allclose(o.smatvec(mu, V[:, 0]), Smu @ V[:, 0], rtol=1e-11, atol=1e-11)
    assert abs(o.inner_C(R, D) - np.sum(Cd * (R @ D.T))) <= 1e-11 * (1 + np.abs(Cd).sum())
    assert abs(o.normC() - np.linalg.norm(Cd)) <= 1e-11 * (1 + np.linalg.norm(Cd))
    # quartic coefficients: dense expansion of f(R + aD)
    q1 = np.array([np.sum(Ai * (R @ D.T + D @ R.T)) for Ai in Ad])
    q2 = np.array([np.sum(Ai * (D @ D.T)) for Ai in Ad])
    pd = [f,
          2 * np.sum(Cd * (R @ D.T)) - y @ q1 + sigma * q @ q1,
          np.sum(Cd * (D @ D.T)) - y @ q2 + 0.5 * sigma * q1 @ q1 + sigma * q @ q2,
          sigma * q1 @ q2, 0.5 * sigma * q2 @ q2]
    np.testing.assert_allclose(o.linesearch(y, sigma, R, D), pd, rtol=1e-10, atol=1e-10)


@pytest.mark.parametrize("idx", [0, 2, 3])
def test_finite_differences_and_quartic(Oracle, idx):
    """grad against central differences; phi(alpha) is *exactly* the quartic; p0 = f, p1 = <G,D>."""
    w = inputs.small(idx)
    o = Oracle(w.problem)
    rng = np.random.default_rng(5)
    G = o.grad(w.y, w.sigma, w.R)
    scale = np.abs(w.R).mean()
    for _ in range(3):
        E = rng.standard_normal(w.R.shape) * scale
        h = 1e-6
        fd = (o.f(w.y, w.sigma, w.R + h * E) - o.f(w.y, w.sigma, w.R - h * E)) / (2 * h)
        assert abs(fd - np.vdot(G, E)) <= 1e-7 * max(1.0, abs(np.vdot(G, E)), np.linalg.norm(G) * np.linalg.norm(E))
    p = o.linesearch(w.y, w.sigma, w.R, w.D)
    assert abs(p[0] - o.f(w.y, w.sigma, w.R)) <= 1e-12 * (1 + abs(p[0]))
    assert abs(p[1] - np.vdot(G, w.D)) <= 1e-10 * (1 + np.abs(p).sum())
    assert p[4] >= 0
    for a in [-1.3, -0.4, 0.25, 0.9, 2.0, 3.7]:
        fa = o.f(w.y, w.sigma, w.R + a * w.D)
        pa = sum(p[k] * a ** k for k in range(5))
        assert abs(fa - pa) <= 1e-11 * sum(abs(p[k]) * abs(a) ** k for k in range(5))


def test_identities(Oracle):
    """adjoint identity, rotation covariance, <C,RR^T> = <G,R>/2 + lambda^T z, MaxCut row norms."""
    rng = np.random.default_rng(11)
    P = random_problem(rng, 40, 60, pC=1)
    o = Oracle(P)
    R = rng.standard_normal((40, 5)); y = rng.standard_normal(60); sigma = 1.3
    w = rng.standard_normal(60)
    P0 = random_problem(rng, 40, 60, nnzC=0)          # C = 0:  (C - A^*(w)) R = -A^*(w) R
    o0 = Oracle(P0)
    assert abs(w @ o0.A_op(R) + np.vdot(R, o0.smatvec(w, R))) <= 1e-11 * (1 + abs(w @ o0.A_op(R)))
    Q, _ = np.linalg.qr(rng.standard_normal((5, 5)))
    np.testing.assert_allclose(o.grad(y, sigma, R @ Q), o.grad(y, sigma, R) @ Q, rtol=1e-10, atol=1e-10)
    assert abs(o.f(y, sigma, R @ Q) - o.f(y, sigma, R)) <= 1e-11 * abs(o.f(y, sigma, R))
    lam, z = o.lam(y, sigma, R)
    G = o.grad(y, sigma, R)
    assert abs(o.inner_C(R, R) - (0.5 * np.vdot(G, R) + lam @ z)) <= 1e-10 * (1 + abs(lam @ z))
    wl = inputs.small(1)
    np.testing.assert_allclose(Oracle(wl.problem).A_op(wl.R), (wl.R ** 2).sum(1), rtol=1e-13)
    # planted right-hand side of config 3 is A(R0 R0^T): generator and oracle agree
    rng3 = inputs._rng(7)
    P3, R0 = inputs.random_sparse_problem(rng3, 500, 900, 4, 1000, 5, f32=False)
    np.testing.assert_allclose(Oracle(P3).A_op(R0), P3.b, rtol=1e-11, atol=1e-14)


# ---------------------------------------------------------------------------------------------
# the paper's worked examples
# ---------------------------------------------------------------------------------------------
def _bp_problem(n, r):
    """(P) of eq. 37; constraints indexed (i,j), 1<=i<=j<=r, row by row."""
    A, b, idx = [], [], {}
    for i in range(r):
        for j in range(i, r):
            idx[(i, j)] = len(A)
            if i < j:
                A.append([(i, j, 0.5)])
            elif i < r - 1:
                A.append([(i, i, 1.0)])
            else:
                A.append([(t, t, 1.0) for t in range(r)])
            b.append(1.0 if (i == j == 0 or i == j == r - 1) else 0.0)
    C = [(t, t, 1.0) for t in range(r, n)]
    return problem_from_lists(n, C, A, b), idx


def test_eq36(Oracle):
    g = GOLD["eq36"]
    P = problem_from_lists(2, [], [[(0, 0, 1.0)], [(0, 1, 0.5)], [(0, 0, 1.0), (1, 1, 1.0)]], g["b"])
    o = Oracle(P)
    y, rho = np.array(g["y"]), g["rho"]
    np.testing.assert_allclose(o.smatvec(y, np.eye(2)), np.diag(g["Z_y_diag"]), atol=1e-15)
    F = np.diag(np.sqrt(g["X_min_diag"]))
    assert abs(o.f(y, rho, F) - g["f_at_min"]) < 1e-15
    assert np.abs(o.grad(y, rho, F)).max() < 1e-15
    lam, _ = o.lam(y, rho, F)
    assert np.abs(o.smatvec(lam, np.eye(2))).max() < 1e-15       # Z(z_{y,rho}) = 0 here
    rng = np.random.default_rng(0)                               # unique minimiser of (AL-P)
    for _ in range(20):
        assert o.f(y, rho, F + 0.3 * rng.standard_normal((2, 2))) > g["f_at_min"]


@pytest.mark.parametrize("n,r", GOLD["eq37_39"]["cases"])
def test_eq37_39(Oracle, n, r):
    P, idx = _bp_problem(n, r)
    o = Oracle(P)
    y = np.zeros(P.m)
    for i in range(r):
        y[idx[(i, i)]] = 1 / (2 * r)
    y[idx[(0, 0)]] = 1 / (2 * r) - 1
    y[idx[(r - 1, r - 1)]] = -0.5
    Zy = np.concatenate([[1.5 - 1 / (2 * r)], np.full(r - 2, 0.5 - 1 / (2 * r)), [0.5], np.ones(n - r)])
    if r == 1:
        Zy = None
    if Zy is not None:
        np.testing.assert_allclose(o.smatvec(y, np.eye(n)), np.diag(Zy), atol=1e-15)
    F = np.zeros((n, r)); F[:r, :r] = np.sqrt(1 / (2 * r)) * np.eye(r)
    assert np.abs(o.grad(y, 1.0, F)).max() < 1e-15
    lam, _ = o.lam(y, 1.0, F)
    np.testing.assert_allclose(o.smatvec(lam, np.eye(n)), np.diag(np.r_[np.zeros(r), np.ones(n - r)]), atol=1e-15)


@pytest.mark.parametrize("n,r,e", GOLD["eq40_41"]["cases"])
def test_eq40_41(Oracle, n, r, e):
    P, idx = _bp_problem(n, r)
    o = Oracle(P)
    y = np.zeros(P.m)
    for i in range(1, r - 1):
        y[idx[(i, i)]] = e
    y[idx[(0, 0)]] = -2 * (r - 1) * e
    y[idx[(r - 1, r - 1)]] = -(r - 1) * e
    Zy = np.r_[3 * (r - 1) * e, np.full(r - 2, (r - 2) * e), (r - 1) * e, np.ones(n - r)]
    np.testing.assert_allclose(o.smatvec(y, np.eye(n)), np.diag(Zy), atol=1e-15)
    F = np.zeros((n, r)); F[:r, :r] = np.diag(np.sqrt(np.r_[1 - 2 * (r - 1) * e, np.full(r - 1, e)]))
    assert np.abs(o.grad(y, 1.0, F)).max() < 1e-14


@pytest.mark.parametrize("eps,rho,delta", GOLD["eq42_43"]["cases"])
def test_eq42_43(Oracle, eps, rho, delta):
    P = problem_from_lists(2, [], [[(0, 0, 1.0)], [(1, 1, 1.0)]], [0.0, 1.0])
    o = Oracle(P)
    y = np.array([-eps, 0.0])
    F = np.array([[np.sqrt(delta)], [1.0]]); Fs = np.array([[0.0], [1.0]])
    assert abs((o.f(y, rho, F) - o.f(y, rho, Fs)) - (eps * delta + rho * delta ** 2 / 2)) < 1e-14


def prop6_instance():
    g = GOLD["prop6"]
    d, k, rho, eta = g["d"], g["k"], g["rho"], g["eta"]
    eps = 0.9 * eta ** 2 * rho / 4
    a = eta ** 2 * k
    A = [[(i, d - 1, 0.5)] for i in range(d - 1)] + [[(i, i, eps) for i in range(d)]]
    C = [(i, i, 2 * eps) for i in range(d - 1)] + [(d - 1, d - 1, eps)]
    P = problem_from_lists(d, C, A, [0.0] * (d - 1) + [eps * a])
    y = np.array([0.0] * (d - 1) + [2.0])
    F = np.zeros((d, k)); F[:k, :k] = eta * np.eye(k)
    return P, y, F, rho, eps, a


def test_prop6(Oracle):
    P, y, F, rho, eps, a = prop6_instance()
    d = P.n
    o = Oracle(P)
    assert np.abs(o.A_op(F) - P.b).max() < 1e-15                       # eq. 66, feasibility
    S = np.zeros((d, d)); S[-1, -1] = -eps
    np.testing.assert_allclose(o.smatvec(y, np.eye(d)), S, atol=1e-15)  # eq. 66, C - A^* y
    assert np.abs(o.grad(y, rho, F)).max() < 1e-15                     # eq. 67
    # growth step along v = e_d: L drops by exactly theta^2 / (2 rho |A(vv^T)|^2) = 1/(2 rho)
    v = np.zeros((d, 1)); v[-1] = 1.0
    av = o.A_op(v)
    s_star = eps / (rho * av @ av)
    assert abs(s_star - 1 / (rho * eps)) < 1e-12
    F2 = np.hstack([F, np.sqrt(s_star) * v])
    assert abs((o.f(y, rho, F) - o.f(y, rho, F2)) - 1 / (2 * rho)) < 1e-12


def test_prop7(Oracle):
    g = GOLD["prop7"]
    d, k, rho, eps = g["d"], g["k"], g["rho"], g["eps"]
    eta2, a = 4 / (eps * k), 7 / eps
    A = [[(i, d - 1, 0.5)] for i in range(d - 1)]
    A.append([(i, i, eps) for i in range(d)])
    A.append([(i, i, 2 * eps) for i in range(d - 1)] + [(d - 1, d - 1, eps)])
    P = problem_from_lists(d, [], A, [0.0] * (d - 1) + [eps * a, eps * a])
    o = Oracle(P)
    y = np.array([0.0] * (d - 1) + [rho, -rho])
    F = np.zeros((d, k)); F[:k, :k] = np.sqrt(eta2) * np.eye(k)
    lam, _ = o.lam(y, rho, F)
    S = np.zeros((d, d)); S[-1, -1] = -2 * eps * rho
    np.testing.assert_allclose(o.smatvec(lam, np.eye(d)), S, atol=1e-13)  # eq. 73
    assert np.abs(o.grad(y, rho, F)).max() < 1e-13                       # eq. 74


def test_appC(Oracle):
    g = GOLD["appC"]
    eps, eta = g["eps"], g["eta"]
    X11 = 1 - (1 - eta) * eps
    X33 = (np.sqrt(1 + 4 * eta * eps * (1 - (1 - eta) * eps)) - 1) / 2
    delta = -(np.sqrt(eta * eps * (1 + X33)) + np.sqrt(X11 * X33))
    P = problem_from_lists(3, [], [[(0, 0, 1.0), (1, 1, 1.0)], [(2, 2, 1.0)], [(0, 2, 1.0)]], [1.0, 0.0, 0.0])
    o = Oracle(P)
    y = np.array([-eps, -1.0, -delta])
    w0 = np.array([[np.sqrt(X11)], [0.0], [np.sqrt(X33)]])
    for xi in g["xis"]:
        w = w0.copy(); w[1, 0] = xi
        assert abs((o.f(y, 1.0, w) - o.f(y, 1.0, w0)) - (xi ** 2 * eta * eps + xi ** 4 / 2)) < 1e-14  # eq. 107


def _graph_maxcut(n, edges):
    lo = np.array([min(e) for e in edges]); hi = np.array([max(e) for e in edges])
    return inputs.maxcut_problem(n, lo, hi, np.ones(len(edges)))


@pytest.mark.parametrize("n", GOLD["maxcut_optima"]["Kn"])
def test_Kn_certificate(Oracle, n):
    """S(y*) = J/4 for y* = -(n/4) 1: lambda_min = 0, and X = (n I - J)/(n-1) attains -n^2/4."""
    P = _graph_maxcut(n, [(i, j) for i in range(n) for j in range(i + 1, n)])
    o = Oracle(P)
    np.testing.assert_allclose(o.smatvec(np.full(n, -n / 4), np.eye(n)), np.full((n, n), 0.25), atol=1e-14)
    X = (n * np.eye(n) - np.ones((n, n))) / (n - 1)
    mu, Q = np.linalg.eigh(X)
    R = Q[:, 1:] * np.sqrt(mu[1:])
    np.testing.assert_allclose(o.A_op(R), np.ones(n), atol=1e-13)
    assert abs(o.inner_C(R, R) + n * n / 4) < 1e-12


@pytest.mark.parametrize("n", GOLD["maxcut_optima"]["Cn"])
def test_Cn_certificate(Oracle, n):
    """Odd cycle: y* = -(1/2)(1+cos(pi/n)) 1 gives lambda_min(S) = 0 with multiplicity 2; the 2-D
    unit vectors at angle pi(n-1)/n attain -(n/2)(1+cos(pi/n))."""
    P = _graph_maxcut(n, [(i, (i + 1) % n) for i in range(n)])
    o = Oracle(P)
    S = o.smatvec(np.full(n, -0.5 * (1 + np.cos(np.pi / n))), np.eye(n))
    ev = np.linalg.eigvalsh(S)
    assert abs(ev[0]) < 1e-13 and abs(ev[1]) < 1e-13 and ev[2] > 1e-6
    ang = np.pi * (n - 1) / n * np.arange(n)
    R = np.c_[np.cos(ang), np.sin(ang)]
    assert abs(o.inner_C(R, R) + n / 2 * (1 + np.cos(np.pi / n))) < 1e-12
