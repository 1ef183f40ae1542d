"""Oracle, Part 2: the ALORA iteration -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Follows Algorithm 1 (section 5) step by step, in the paper's order.  ALORA is a
heuristic without a closed-form result, so this file *is* the definition the CUDA library's
``alora_solve`` / ``alora_lanczos`` are compared with.  Wherever the paper is silent the reading of
DESIGN.md ("Readings", numbers in brackets below = SURVEY.md section 8c) is taken; every free
constant is a field of ``Params`` with the same default as ``alora_params`` in include/alora.h.

Library primitives used as steps: numpy dot/matmul, ``numpy.roots`` (cubic), ``numpy.linalg.eigh``
(r x r), ``scipy.linalg.eigh_tridiagonal`` (Lanczos tridiagonal).

parity unpinned (by the paper): the L-BFGS / sigma-schedule / shrink constants are free parameters
(readings 5, 6, 12, 13); they are pinned only oracle-vs-GPU.  What *is* pinned against the paper
and mathematics (tests/test_oracle_alm.py): closed-form MaxCut / theta optima, Prop. 6 escape,
Lanczos against a dense eigen-solver, exact line search against a brute-force scan, the matrix-completion
optimum against the nuclear norm (SVD), the p_max > 1 growth step against its model identity (exact decrease
of the augmented Lagrangian), the KKT conditions of the small SDP and the p = 1 closed form.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np
from scipy.linalg import eigh_tridiagonal


@dataclass
class Params:
    eps: float = 1e-5          # KKT tolerance, eq. 77
    stop_mode: int = 0         # 0: all three terms of eq. 77 <= eps; 1: primal infeasibility term only
    T_max: int = 100           # outer iterations
    tol0: float = 1e-2         # [6] inner tolerance: tol_t = max(tol_min, min(tol0, c_in * infeas_{t-1}))
    c_in: float = 0.1
    tol_min: float = 1e-7
    it_max: int = 500          # [6] inner iterations per outer iteration
    lbfgs_mem: int = 5         # [5] 0 = steepest descent with exact step (the paper's GD)
    p_max: int = 1             # [7, 29] eigenvectors per growth step (1: closed form; up to 4: small SDP)
    tau_neg: float = -1.0      # [8] growth threshold; < 0 means "use eps"
    tol_eig: float = -1.0      # [9] Lanczos residual tolerance; < 0 means eps/10
    k_max: int = 300           # [9] Lanczos steps
    gamma: float = 2.0         # [12] sigma <- min(gamma sigma, sigma_max) if ||q|| > kappa ||q_prev|| and kkt[0] > eps
    kappa: float = 0.25
    sigma_max: float = 1e8
    tau_shrink: float = 1e-8   # [13] drop directions of R^T R with mu_j <= tau_shrink * mu_max
    s_max: float = 1e6         # [7] cap of the growth step when A(vv^T) = 0
    seed: int = 12345          # Lanczos start vectors: counter_uniform(seed + run index, i)
    stall_tol: float = 0.0     # [28] inner loop also stops after stall_iters consecutive steps whose predicted
    stall_iters: int = 3       #      decrease phi(0) - phi(alpha) <= stall_tol (1 + |f|); 0 = off


def preset_params(f32: bool, **kw) -> Params:
    """Same preset as alora_preset_params (include/alora.h): fp32 storage -> bounded inexact inner solves
    (it_max = 100) with the stall rule [28] on."""
    base = dict(it_max=100, stall_tol=1e-9, stall_iters=3) if f32 else {}
    base.update(kw)
    return Params(**base)


@dataclass
class IterRecord:
    t: int = 0
    r: int = 0
    sigma: float = 0.0
    cx: float = 0.0            # <C, RR^T> after the inner solve
    f: float = 0.0
    qnorm: float = 0.0         # ||A(RR^T) - b|| at the dual update
    gnorm: float = 0.0
    theta1: float = 0.0        # smallest Ritz value of S(lambda)
    inner_iters: int = 0
    n_evals: int = 0
    lanczos_steps: int = 0
    grew: int = 0
    shrank: int = 0
    kkt: tuple = (0.0, 0.0, 0.0)


@dataclass
class Result:
    R: np.ndarray = None
    y: np.ndarray = None
    sigma: float = 0.0
    converged: bool = False
    outer_iters: int = 0
    n_evals: int = 0
    n_linesearch: int = 0
    n_matvec: int = 0
    kkt: tuple = (0.0, 0.0, 0.0)
    log: list = field(default_factory=list)


# ---------------------------------------------------------------------------------------------
def counter_uniform(seed: int, count: int) -> np.ndarray:
    """v[i] in (-1,1) from a splitmix64-style hash of (seed, i): integer arithmetic only, so the
    CUDA side (its own implementation) produces the same bits  [9]."""
    with np.errstate(over="ignore"):
        x = np.arange(count, dtype=np.uint64) + np.uint64(seed) * np.uint64(0x9E3779B97F4A7C15)
        x = (x ^ (x >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)
        x = (x ^ (x >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)
        x = x ^ (x >> np.uint64(31))
    return ((x >> np.uint64(11)).astype(np.float64) + 0.5) * (2.0 / 9007199254740992.0) - 1.0


def quartic_argmin(p) -> tuple[float, int]:
    """Exact line search [20]: minimiser over alpha > 0 of phi(alpha) = sum_k p_k alpha^k.

    Real roots of phi'(alpha) = p1 + 2 p2 alpha + 3 p3 alpha^2 + 4 p4 alpha^3, two Newton polish
    steps, then the positive root with the smallest phi (ties to rel. 1e-14 -> smallest alpha).
    Returns (alpha, flag); flag = 1 when no positive stationary point exists (alpha = 1 returned).
    """
    p0, p1, p2, p3, p4 = (float(v) for v in p)
    if p4 == 0.0 and p3 == 0.0:
        if p2 > 0.0 and -p1 / (2.0 * p2) > 0.0:
            return -p1 / (2.0 * p2), 0
        return 1.0, 1
    roots = np.roots([4.0 * p4, 3.0 * p3, 2.0 * p2, p1])
    scale = max(1.0, float(np.max(np.abs(roots)))) if roots.size else 1.0
    cand = []
    for z in roots:
        if abs(z.imag) <= 1e-8 * scale:
            a = float(z.real)
            for _ in range(2):  # Newton on phi'
                d1 = p1 + a * (2 * p2 + a * (3 * p3 + a * 4 * p4))
                d2 = 2 * p2 + a * (6 * p3 + a * 12 * p4)
                if d2 != 0.0:
                    a -= d1 / d2
            if a > 0.0:
                cand.append(a)
    if not cand:
        return 1.0, 1
    cand.sort()
    phi = lambda a: p0 + a * (p1 + a * (p2 + a * (p3 + a * p4)))
    best = cand[0]
    for a in cand[1:]:
        if phi(a) < phi(best) - 1e-14 * (abs(phi(best)) + abs(p0)):
            best = a
    return best, 0


def lanczos(matvec, n: int, seed: int, k_max: int, tol_abs: float, p_want: int = 1):
    """Smallest Ritz pair of a symmetric operator by Lanczos with full re-orthogonalisation
    (two passes of classical Gram-Schmidt) [9].  Stops at step k when the residual estimate
    |beta_k s_k| of the smallest Ritz pair is <= tol_abs, on breakdown (beta_k ~ 0), or k = k_max.
    Returns (theta, v, k_used, resid); with p_want > 1 a fifth item (thetas, U): the min(p_want, k)
    smallest Ritz values of the same k-step tridiagonal, ascending, and their unit Ritz vectors as
    columns (the Rayleigh quotient of a Ritz vector IS its Ritz value, converged or not) [29]."""
    v = counter_uniform(seed, n)
    v /= np.sqrt(v @ v)
    V = np.zeros((min(k_max, n), n))
    alphas, betas = [], []
    theta, s, resid = 0.0, np.ones(1), np.inf
    k = 0
    while True:
        V[k] = v
        w = matvec(v)
        a = float(v @ w)
        alphas.append(a)
        w = w - a * v - (betas[-1] * V[k - 1] if k > 0 else 0.0)
        for _ in range(2):
            w = w - V[: k + 1].T @ (V[: k + 1] @ w)
        beta = float(np.sqrt(w @ w))
        k += 1
        if k == 1:
            theta, s = alphas[0], np.ones(1)
        else:
            th, S = eigh_tridiagonal(np.array(alphas), np.array(betas), select="i", select_range=(0, 0))
            theta, s = float(th[0]), S[:, 0]
        resid = abs(beta * s[-1])
        tnorm = max(abs(x) for x in alphas + betas + [1e-300])
        if resid <= tol_abs or beta <= 1e-14 * tnorm or k >= min(k_max, n):
            break
        betas.append(beta)
        v = w / beta
    ritz = V[:k].T @ s
    ritz /= np.sqrt(ritz @ ritz)
    if p_want <= 1:
        return theta, ritz, k, resid
    if k == 1:
        return theta, ritz, k, resid, (np.array([theta]), ritz[:, None])
    pw = min(p_want, k)
    th, S = eigh_tridiagonal(np.array(alphas), np.array(betas[: k - 1]), select="i", select_range=(0, pw - 1))
    U = V[:k].T @ S
    U /= np.sqrt((U * U).sum(axis=0))
    return theta, ritz, k, resid, (th, U)


def psd_project(S):
    """Nearest positive semidefinite matrix in Frobenius norm (eigenvalue clipping)."""
    mu, Q = np.linalg.eigh(0.5 * (S + S.T))
    return (Q * np.maximum(mu, 0.0)) @ Q.T


def growth_sdp(theta, H, sigma: float, iters: int = 500):
    """Alg. 1 line 7 for p negative-curvature directions U = [v_1 .. v_p] with Rayleigh
    quotients theta (U^T S(lambda) U = diag(theta) for Ritz vectors of one Krylov space):
        min_{S >= 0}  g(S) = sum_a theta_a S_aa + (sigma/2) || sum_{a<=b} w_ab S_ab c_ab ||^2,
    c_ab = A((v_a v_b^T + v_b v_a^T)/2), w_ab = 1 (a = b) or 2, H[(ab),(cd)] = <c_ab, c_cd> with the pairs
    a <= b in row-major order.  g(S) is exactly L_rho(X + U S U^T, y) - L_rho(X, y) (expand (AL)).
    Projected gradient with step 1/L from S0 = diag(-theta_a / (sigma H[(aa),(aa)])) [10, 29].
    Returns (S, g(S))."""
    p = len(theta)
    pairs = [(a, b) for a in range(p) for b in range(a, p)]
    wgt = np.array([1.0 if a == b else 2.0 for a, b in pairs])
    Hw = H * np.outer(wgt, wgt)

    def vec(S):
        return np.array([S[a, b] for a, b in pairs])

    def g(S):
        s = vec(S)
        return float(theta @ np.diag(S) + 0.5 * sigma * s @ Hw @ s)

    def grad(S):
        t = sigma * (Hw @ vec(S))          # d/ds of the quadratic term
        G = np.zeros((p, p))
        for (a, b), tv in zip(pairs, t):
            if a == b:
                G[a, a] = tv
            else:
                G[a, b] = G[b, a] = 0.5 * tv   # s_ab stands for the two entries S_ab = S_ba
        return G + np.diag(theta)

    # Lipschitz constant of grad in the Frobenius metric of S: sigma * lambda_max of the quadratic form in S-entries
    D = np.diag([1.0 if a == b else 1.0 / np.sqrt(2.0) for a, b in pairs])
    L = sigma * max(np.linalg.eigvalsh(D @ Hw @ D)[-1], 1e-300)
    S = np.diag([(-theta[a] / (sigma * H[pairs.index((a, a)), pairs.index((a, a))]))
                 if H[pairs.index((a, a)), pairs.index((a, a))] > 0 else 0.0 for a in range(p)])
    S = np.maximum(S, 0.0)
    for _ in range(iters):
        S = psd_project(S - grad(S) / L)
    return S, g(S)


def lbfgs_direction(G, S_list, Y_list):
    """Two-loop recursion: D = -H G with H the L-BFGS inverse-Hessian built from the stored
    (s, y) pairs, initial scaling s^T y / y^T y of the newest pair  [5]."""
    q = G.copy()
    al = []
    for s, yv in zip(reversed(S_list), reversed(Y_list)):
        rho = 1.0 / float(np.vdot(yv, s))
        a = rho * float(np.vdot(s, q))
        al.append(a)
        q -= a * yv
    if S_list:
        q *= float(np.vdot(S_list[-1], Y_list[-1])) / float(np.vdot(Y_list[-1], Y_list[-1]))
    for (s, yv), a in zip(zip(S_list, Y_list), reversed(al)):
        rho = 1.0 / float(np.vdot(yv, s))
        be = rho * float(np.vdot(yv, q))
        q += (a - be) * s
    return -q


def kkt_terms(qnorm, normb, theta_min, normC, cx, by):
    """The three terms of eq. 77."""
    return (qnorm / (1.0 + normb),
            abs(min(0.0, theta_min)) / (1.0 + normC),
            abs(cx - by) / (1.0 + abs(cx) + abs(by)))


def kkt_at(orc, R, y, theta_min):
    """KKT(X, y) of eq. 77 at X = RR^T, from the definitions: ||A(X) - b||_2, ||b||_2,
    ||C||_F, <C,X>, b^T y (l2 norms); theta_min = lambda_min(C - A^*(y)) is passed in
    (the loop has it from Lanczos [16], the pins from a dense eigen-solver)."""
    b = orc.b
    q = orc.A_op(R) - b
    return kkt_terms(float(np.sqrt(q @ q)), float(np.sqrt(b @ b)), theta_min, orc.normC(),
                     orc.inner_C(R, R), float(b @ y))


def shrink_rank(R, tau_shrink: float):
    """Rank shrink [13]: eigen-decompose R^T R = Q M Q^T and drop the directions with
    mu_j <= tau_shrink * mu_max, R <- R Q_keep.  X = RR^T loses only the dropped directions' mu_j, so with
    exact null directions X (hence f, A(X), ||G||_F) is unchanged.  Returns (R_new, number dropped);
    never drops everything."""
    mu, Q = np.linalg.eigh(R.T @ R)
    keep = mu > tau_shrink * mu[-1]
    if not keep.all() and keep.any():
        return R @ Q[:, keep], int((~keep).sum())
    return R, 0


def solve(orc, R0, y0, sigma0: float, prm: Params = Params()) -> Result:
    """ALORA (Algorithm 1) with readings 5-13, 17, 20 of DESIGN.md.

    orc: oracle.Oracle for the problem.  R0: n x r0 start, y0: start dual (paper: 0).
    """
    n = orc.n
    b = orc.b
    tau_neg = prm.tau_neg if prm.tau_neg >= 0 else prm.eps
    tol_eig = prm.tol_eig if prm.tol_eig >= 0 else prm.eps / 10.0
    normC, normb = orc.normC(), float(np.sqrt(b @ b))
    R, y, sigma = np.array(R0, float), np.array(y0, float), float(sigma0)
    res = Result()
    infeas_prev, qnorm_prev, run = np.inf, np.inf, 0

    def run_lanczos(w, p_want=1):
        nonlocal run
        def mv(v):
            res.n_matvec += 1
            return orc.smatvec(w, v)
        out = lanczos(mv, n, prm.seed + run, prm.k_max, tol_eig * (1.0 + normC), p_want)
        run += 1
        return out

    for t in range(prm.T_max):
        rec = IterRecord(t=t, sigma=sigma)
        # -- 1. inner solve: F <- argmin_F L_rho(FF^T, y)            (Alg. 1 line 4)
        tol_t = max(prm.tol_min, min(prm.tol0, prm.c_in * infeas_prev))
        S_list, Y_list = [], []
        it, D, alpha, G_prev, stalled = 0, None, 0.0, None, 0
        while True:
            G = orc.grad(y, sigma, R)
            rec.n_evals += 1
            gnorm = float(np.sqrt(np.vdot(G, G)))
            if G_prev is not None and prm.lbfgs_mem > 0:
                s, yv = alpha * D, G - G_prev
                sy, ss, yy = float(np.vdot(s, yv)), float(np.vdot(s, s)), float(np.vdot(yv, yv))
                if sy > 1e-10 * np.sqrt(ss * yy):
                    S_list.append(s); Y_list.append(yv)
                    if len(S_list) > prm.lbfgs_mem:
                        S_list.pop(0); Y_list.pop(0)
            if gnorm / (1.0 + normC) <= tol_t or it >= prm.it_max:
                break
            D = lbfgs_direction(G, S_list, Y_list) if S_list else -G
            if float(np.vdot(G, D)) >= 0.0:        # not a descent direction: restart from -G
                S_list, Y_list, D = [], [], -G
            p = orc.linesearch(y, sigma, R, D)     # quartic coefficients of f(R + alpha D)
            res.n_linesearch += 1
            alpha, _ = quartic_argmin(p)
            if prm.stall_tol > 0.0:
                dec = -alpha * (p[1] + alpha * (p[2] + alpha * (p[3] + alpha * p[4])))
                stalled = stalled + 1 if dec <= prm.stall_tol * (1.0 + abs(p[0])) else 0
                if stalled >= prm.stall_iters:
                    break
            G_prev = G
            R = R + alpha * D
            it += 1
        rec.inner_iters, rec.gnorm = it, gnorm
        rec.f = orc.f(y, sigma, R)
        # -- 2. q = A(RR^T) - b,  lambda = y - sigma q
        lam, z = orc.lam(y, sigma, R)
        q = z - b
        # -- 3. eigenvector of nabla_X L_rho = C - A^*(lambda)         (Alg. 1 line 5)
        multi = None
        if prm.p_max > 1:
            theta, v, ksteps, _, multi = run_lanczos(lam, prm.p_max)
        else:
            theta, v, ksteps, _ = run_lanczos(lam)
        rec.theta1, rec.lanczos_steps = theta, ksteps
        theta_kkt, changed = theta, False
        if -theta / (1.0 + normC) > tau_neg:
            # -- 4. grow: S <- argmin_{S>=0} L_rho(FF^T + V S V^T, y), F <- [F, V S^{1/2}]
            #       (Alg. 1 lines 6-8)
            cols = None
            if multi is not None:
                # [29] every Ritz pair of the run that is itself sufficiently negative joins V
                ths, U = multi
                sel = [j for j in range(len(ths)) if -ths[j] / (1.0 + normC) > tau_neg]
                if len(sel) > 1:
                    U, ths = U[:, sel], ths[sel]
                    pairs = [(a, c) for a in range(len(sel)) for c in range(a, len(sel))]
                    cab = np.array([orc.A_sym(U[:, [a]], U[:, [c]]) for a, c in pairs])
                    S, gval = growth_sdp(ths, cab @ cab.T, sigma)
                    if gval < 0.0:
                        mu, Q = np.linalg.eigh(S)
                        keep = mu > 1e-12 * mu[-1]
                        cols = U @ (Q[:, keep] * np.sqrt(mu[keep]))      # [11] V S^{1/2} with S^{1/2} = Q mu^{1/2}
            if cols is None:
                # p = 1 closed form: L(X + s vv^T) - L(X) = s theta + (sigma/2) s^2 ||A(vv^T)||^2
                av = orc.A_op(v[:, None])
                den = sigma * float(av @ av)
                s_star = -theta / den if den > 0.0 and -theta / den < prm.s_max else prm.s_max
                cols = np.sqrt(s_star) * v[:, None]
            R = np.hstack([R, cols])
            rec.grew, changed = cols.shape[1], True
        elif R.shape[1] > 1:
            # -- 5. shrink [13]: drop the numerically null directions of R
            R, dropped = shrink_rank(R, prm.tau_shrink)
            if dropped:
                rec.shrank, changed = dropped, True
        if changed:
            q = orc.A_op(R) - b
        qnorm = float(np.sqrt(q @ q))
        # -- 6. y <- y + rho (b - A FF^T)                              (Alg. 1 line 10)
        y = y - sigma * q
        if changed:                       # [17] S(lambda) != S(y_new) once R changed: recompute
            theta_kkt, _, _, _ = run_lanczos(y)
        cx = orc.inner_C(R, R)
        rec.kkt = kkt_at(orc, R, y, theta_kkt)        # eq. 77 at (RR^T, y_new)
        rec.r, rec.cx, rec.qnorm = R.shape[1], cx, qnorm
        # -- 7. sigma schedule [12]
        if qnorm > prm.kappa * qnorm_prev and rec.kkt[0] > prm.eps:   # no increase once the primal term is below eps
            sigma = min(prm.gamma * sigma, prm.sigma_max)
        qnorm_prev, infeas_prev = qnorm, rec.kkt[0]
        res.log.append(rec)
        res.n_evals += rec.n_evals
        # -- 8. until KKT(FF^T, y) <= eps                              (Alg. 1 line 11, eq. 77)
        done = rec.kkt[0] <= prm.eps if prm.stop_mode == 1 else max(rec.kkt) <= prm.eps
        if done:
            res.converged = True
            break
    res.R, res.y, res.sigma = R, y, sigma
    res.outer_iters, res.kkt = len(res.log), res.log[-1].kkt
    return res
