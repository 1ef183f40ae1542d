"""GPU: Lanczos and the ALORA loop (alora_lanczos / alora_solve) against the oracle's Part 2
(oracle/alm.py) and against closed forms.  Trajectory parity on config 0 follows DESIGN.md
reading 23: same outer iterations, same grow / shrink decisions and ranks; per outer iteration
<C,X>, ||q||/(1+||b||), sigma and theta_1 agree to 1e-6; inner iteration counts within 10 %."""
import numpy as np
import pytest

from paper_2505_15775_b200 import inputs
from tests.test_oracle_pins import _graph_maxcut, prop6_instance

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def torch():
    import torch
    assert torch.cuda.is_available()
    return torch


@pytest.fixture(scope="module")
def binding():
    from paper_2505_15775_b200 import binding
    return binding


@pytest.fixture(scope="module")
def alm():
    from oracle import alm
    return alm


def gpu_solve(torch, binding, P, dtype, R0, y0, sigma, r_cap, **kw):
    tdt = torch.float32 if dtype == inputs.F32 else torch.float64
    ctx = binding.Context(P, dtype)
    n, r0 = R0.shape
    Rbuf = torch.zeros(n * r_cap, dtype=tdt, device="cuda")
    Rbuf[: n * r0] = torch.as_tensor(np.ascontiguousarray(R0), dtype=tdt).cuda().reshape(-1)
    y = torch.as_tensor(np.ascontiguousarray(y0), dtype=torch.float64).cuda()
    res, log, r, sg, ok = ctx.solve(binding.Params(**kw), Rbuf, r0, r_cap, y, sigma)
    R = Rbuf[: n * r].reshape(n, r).cpu().numpy().astype(float)
    out = dict(res=res, log=log, r=r, sigma=sg, ok=ok, R=R, y=y.cpu().numpy())
    ctx.close()
    return out


def test_lanczos_matches_oracle_and_dense(torch, binding, alm, oracle_mod):
    w = inputs.small(0)
    P = w.problem
    o = oracle_mod.Oracle(P)
    mu = np.random.default_rng(1).standard_normal(P.m)
    S = o.smatvec(mu, np.eye(P.n))
    ev = np.linalg.eigvalsh(S)
    th_o, v_o, k_o, res_o = alm.lanczos(lambda x: o.smatvec(mu, x), P.n, 42, 300, 1e-8)
    ctx = binding.Context(P, inputs.F64)
    mud = torch.as_tensor(mu).cuda()
    v = torch.zeros(P.n, dtype=torch.float64, device="cuda")
    th, k, resid, ok = ctx.lanczos(mud, 300, 1e-8, 42, v)
    assert ok and abs(th - ev[0]) < 1e-8 and abs(th - th_o) < 1e-9
    assert abs(k - k_o) <= 2
    vv = v.cpu().numpy()
    assert abs(np.linalg.norm(vv) - 1) < 1e-12 and np.linalg.norm(S @ vv - th * vv) < 1e-6
    # iteration cap: ENOTCONV with the best pair so far
    th2, k2, _, ok2 = ctx.lanczos(mud, 5, 1e-12, 42, None)
    assert not ok2 and k2 == 5 and th2 >= ev[0] - 1e-12
    ctx.close()
    # breakdown (two distinct eigenvalues): exact after 2 steps
    P6, y6, F, rho, eps, a = prop6_instance()
    ctx = binding.Context(P6, inputs.F64)
    th, k, resid, ok = ctx.lanczos(torch.as_tensor(y6).cuda(), 50, 1e-12, 1, None)
    assert ok and k == 2 and abs(th + eps) < 1e-14
    ctx.close()


def test_lanczos_multi_pair_abi(torch, binding, alm, oracle_mod):
    """alora_lanczos with p_want = 4 (Alg. 1 line 5): theta ascending, column-major unit Ritz vectors
    with Rayleigh quotients theta (V^T S V = diag(theta)), residual estimates, same values as the oracle's run;
    mu = NULL takes lambda of the last evaluation."""
    w = inputs.small(0)
    P = w.problem
    o = oracle_mod.Oracle(P)
    y = np.random.default_rng(1).standard_normal(P.m)
    lam, _ = o.lam(y, 1.0, w.R)
    S = o.smatvec(lam, np.eye(P.n))
    th_o, v_o, k_o, res_o, (ths_o, U_o) = alm.lanczos(lambda x: o.smatvec(lam, x), P.n, 42, 300, 1e-8, p_want=4)
    ctx = binding.Context(P, inputs.F64)
    Vd = torch.zeros(4 * P.n, dtype=torch.float64, device="cuda")
    ths, k, resid, ok = ctx.lanczos(torch.as_tensor(lam).cuda(), 300, 1e-8, 42, Vd, p_want=4)
    assert ok and ths.shape == (4,) and resid.shape == (4,) and abs(k - k_o) <= 2
    assert np.all(np.diff(ths) >= 0) and np.abs(ths - ths_o).max() < 1e-8 and resid[0] <= 1e-8
    U = Vd.cpu().numpy().reshape(4, P.n).T
    np.testing.assert_allclose(U.T @ U, np.eye(4), atol=1e-9)
    np.testing.assert_allclose(U.T @ S @ U, np.diag(ths), atol=1e-7)
    for j in range(4):     # the residual estimate |beta_k s_kj| is the true residual norm of the Ritz pair
        assert abs(np.linalg.norm(S @ U[:, j] - ths[j] * U[:, j]) - resid[j]) <= 1e-6 * (1 + resid[j])
    # mu = NULL after an evaluation with the same (y, sigma): same operator
    R = torch.as_tensor(w.R).cuda(); yd = torch.as_tensor(y).cuda()
    ctx.set_dual(yd, 1.0)
    with pytest.raises(binding.AloraError) as e:
        ctx.lanczos(None, 300, 1e-8, 42, None)
    assert e.value.status == binding.ESTATE
    ctx.eval(R, w.r, w.r, None, None)
    th1, k1, _, ok1 = ctx.lanczos(None, 300, 1e-8, 42, None)
    assert ok1 and abs(th1 - ths[0]) < 1e-9
    # values only (no vectors), fewer steps than pairs asked for
    th2, k2, r2, ok2 = ctx.lanczos(None, 3, 1e-14, 42, None, p_want=8)
    assert k2 == 3 and th2.shape == (3,) and not ok2
    ctx.close()


def test_lanczos_fp32(torch, binding, oracle_mod):
    w = inputs.small(4)
    P = w.problem
    o = oracle_mod.Oracle(P)
    lam, _ = o.lam(w.y, w.sigma, w.R)
    ctx = binding.Context(P, inputs.F32)
    v = torch.zeros(P.n, dtype=torch.float32, device="cuda")
    th, k, resid, ok = ctx.lanczos(torch.as_tensor(lam).cuda(), 300, 1e-4, 7, v)
    vv = v.cpu().numpy().astype(float)
    Sv = o.smatvec(lam, vv)
    assert abs(vv @ Sv - th) < 1e-4 and np.linalg.norm(Sv - th * vv) < 5e-3
    import scipy.sparse.linalg as sla
    op = sla.LinearOperator((P.n, P.n), matvec=lambda x: o.smatvec(lam, x), dtype=float)
    ref = sla.eigsh(op, k=1, which="SA", tol=1e-8)[0][0]
    assert abs(th - ref) < 1e-3
    ctx.close()


def test_config0_trajectory(torch, binding, alm, oracle_mod):
    w = inputs.full(0)
    o = oracle_mod.Oracle(w.problem)
    ref = alm.solve(o, w.R, w.y, w.sigma, alm.Params(eps=1e-6))
    out = gpu_solve(torch, binding, w.problem, w.dtype, w.R, w.y, w.sigma, r_cap=64, eps=1e-6)
    assert out["ok"] and ref.converged
    assert out["res"].outer_iters == ref.outer_iters
    for a, b in zip(out["log"], ref.log):
        assert (a.r, a.grew, a.shrank) == (b.r, b.grew, b.shrank), (a.t, a.r, b.r)
        assert a.sigma == b.sigma
        assert abs(a.cx - b.cx) <= 1e-6 * abs(b.cx), (a.t, a.cx, b.cx)
        assert abs(a.kkt[0] - b.kkt[0]) <= 1e-6 * max(1e-3, b.kkt[0]) + 1e-9
        assert abs(a.theta1 - b.theta1) <= 1e-6
        assert abs(a.inner_iters - b.inner_iters) <= max(2, 0.1 * b.inner_iters), (a.t, a.inner_iters, b.inner_iters)
    assert max(out["res"].kkt) <= 1e-6
    assert abs(o.inner_C(out["R"], out["R"]) - o.inner_C(ref.R, ref.R)) <= 1e-6 * abs(o.inner_C(ref.R, ref.R))
    np.testing.assert_allclose(out["y"], ref.y, atol=1e-5)


@pytest.mark.parametrize("n", [9, 20])
def test_solve_Kn(torch, binding, oracle_mod, n):
    P = _graph_maxcut(n, [(i, j) for i in range(n) for j in range(i + 1, n)])
    R0 = inputs._unit_rows(np.random.default_rng(n), n, 4)
    out = gpu_solve(torch, binding, P, inputs.F64, R0, np.zeros(n), 1.0, r_cap=32, eps=1e-7)
    o = oracle_mod.Oracle(P)
    assert out["ok"] and abs(o.inner_C(out["R"], out["R"]) + n * n / 4) < 1e-4
    assert np.abs(out["y"] + n / 4).max() < 1e-4


def test_solve_theta_C5(torch, binding, oracle_mod):
    P = inputs.theta_problem(5, np.arange(5), (np.arange(5) + 1) % 5) if False else \
        inputs.theta_problem(5, np.array([0, 1, 2, 3, 0]), np.array([1, 2, 3, 4, 4]))
    R0 = np.random.default_rng(5).standard_normal((5, 3)) / np.sqrt(15)
    out = gpu_solve(torch, binding, P, inputs.F64, R0, np.zeros(P.m), 1.0, r_cap=16, eps=1e-7)
    o = oracle_mod.Oracle(P)
    assert out["ok"] and abs(o.inner_C(out["R"], out["R"]) + np.sqrt(5)) < 1e-4


def test_prop6_escape(torch, binding, oracle_mod):
    """Rank adaptation pass/fail: from the spurious minimiser the solver must grow
    along e_d and reach X* = a e_d e_d^T; with growth disabled it stays put."""
    P, y, F, rho, eps, a = prop6_instance()
    out = gpu_solve(torch, binding, P, inputs.F64, F, y, rho, r_cap=16, gamma=1.0, eps=1e-8)
    assert out["ok"] and out["log"][0].grew == 1 and out["log"][0].inner_iters == 0
    X = out["R"] @ out["R"].T
    Xs = np.zeros((P.n, P.n)); Xs[-1, -1] = a
    assert np.abs(X - Xs).max() < 1e-5
    assert np.abs(out["y"] - np.r_[np.zeros(P.n - 1), 1.0]).max() < 1e-5
    stuck = gpu_solve(torch, binding, P, inputs.F64, F, y, rho, r_cap=16, gamma=1.0, eps=1e-8, tau_neg=1e30, T_max=20)
    assert not stuck["ok"] and all(r.inner_iters == 0 for r in stuck["log"])


def test_solve_fp32_ring_matchings(torch, binding, oracle_mod):
    """Scaled-down config 4 (fp32 R): full rank-adaptive solve to relative primal infeasibility 1e-5."""
    w = inputs.small(4)
    out = gpu_solve(torch, binding, w.problem, w.dtype, w.R, w.y, w.sigma, r_cap=32, eps=1e-5, stop_mode=1)
    assert out["ok"] and out["res"].kkt[0] <= 1e-5
    o = oracle_mod.Oracle(w.problem)
    q = o.A_op(out["R"]) - w.problem.b
    assert np.linalg.norm(q) / (1 + np.linalg.norm(w.problem.b)) <= 2e-5


def test_solve_lbfgs_memory_bounds(torch, binding, oracle_mod):
    """lbfgs_mem = 16 (the documented maximum; the two-loop path, mem >= 8) and a value above it (clamped) reach
    the K_9 optimum; the workspace holds 5 + 2 (16 + 1) arrays."""
    n = 9
    P = _graph_maxcut(n, [(i, j) for i in range(n) for j in range(i + 1, n)])
    R0 = inputs._unit_rows(np.random.default_rng(4), n, 4)
    o = oracle_mod.Oracle(P)
    for mem in (16, 40, 0):
        out = gpu_solve(torch, binding, P, inputs.F64, R0, np.zeros(n), 1.0, r_cap=16, eps=1e-7, lbfgs_mem=mem)
        assert out["ok"] and abs(o.inner_C(out["R"], out["R"]) + n * n / 4) < 1e-4, mem


def test_config4_full_solve(torch, binding, oracle_mod):
    """BASELINE.json's target: the full rank-adaptive ALM solve of the n = 2^24 MaxCut config reaches relative primal
    infeasibility <= 1e-5 (first term of eq. 77) on one B200, with the library's preset for fp32
    contexts (alora_preset_params).  The residual A(RR^T) - b of the returned R is recomputed by the oracle."""
    w = inputs.full(4)
    P = w.problem
    r_cap = w.r + 14
    ctx = binding.Context(P, w.dtype)
    Rbuf = torch.zeros(P.n * r_cap, dtype=torch.float32, device="cuda")
    Rbuf[: P.n * w.r] = torch.as_tensor(w.R, dtype=torch.float32).cuda().reshape(-1)
    y = torch.zeros(P.m, dtype=torch.float64, device="cuda")
    prm = binding.Params.preset(w.dtype, eps=1e-5, stop_mode=1)
    res, log, r, sg, ok = ctx.solve(prm, Rbuf, w.r, r_cap, y, w.sigma)
    assert ok and res.kkt[0] <= 1e-5, (res.kkt[0], res.outer_iters)
    R = Rbuf[: P.n * r].reshape(P.n, r).cpu().numpy().astype(float)
    ctx.close()
    del Rbuf
    o = oracle_mod.Oracle(P)
    q = o.A_op(R) - P.b
    assert np.linalg.norm(q) / (1 + np.linalg.norm(P.b)) <= 1.05e-5
    assert res.seconds < 120.0


def test_rank_cap_skips_growth(torch, binding, oracle_mod):
    """r_cap reached: the growth step is skipped instead of failing (reading 27).  K_9 from rank 1
    with r_cap = 1 cannot reach the optimum (it needs rank >= 2 ... 8), but the call must return cleanly."""
    n = 9
    P = _graph_maxcut(n, [(i, j) for i in range(n) for j in range(i + 1, n)])
    R0 = inputs._unit_rows(np.random.default_rng(3), n, 1)
    out = gpu_solve(torch, binding, P, inputs.F64, R0, np.zeros(n), 1.0, r_cap=1, eps=1e-7, T_max=8)
    assert all(rec.r == 1 and rec.grew == 0 for rec in out["log"])
    # and with room to grow the same start reaches -n^2/4
    out = gpu_solve(torch, binding, P, inputs.F64, R0, np.zeros(n), 1.0, r_cap=16, eps=1e-7)
    o = oracle_mod.Oracle(P)
    assert out["ok"] and abs(o.inner_C(out["R"], out["R"]) + n * n / 4) < 1e-4


@pytest.mark.parametrize("dtype,tol", [(inputs.F64, 1e-5), (inputs.F32, 2e-3)])
def test_solve_matrix_completion(torch, binding, oracle_mod, dtype, tol):
    """Matrix completion: exact recovery of M = U V^T and optimal value = nuclear norm."""
    rng = np.random.default_rng(11)
    n1 = n2 = 20
    P, U, V = inputs.matrix_completion_problem(rng, n1, n2, 2, 300)
    M = U @ V.T
    R0 = rng.standard_normal((P.n, 4))
    out = gpu_solve(torch, binding, P, dtype, R0, np.zeros(P.m), 1.0, r_cap=16,
                    eps=1e-7 if dtype == inputs.F64 else 1e-4)
    assert out["ok"]
    X = out["R"] @ out["R"].T
    assert np.linalg.norm(X[:n1, n1:] - M) <= 10 * tol * np.linalg.norm(M)
    nuc = np.linalg.svd(M, compute_uv=False).sum()
    assert abs(0.5 * np.trace(X) - nuc) <= tol * nuc


def test_solve_pmax3(torch, binding, alm, oracle_mod):
    """p_max = 3 (reading 29): same optimum as the oracle's p_max = 3 and p_max = 1 runs on MaxCut
    G(60,150) from rank 1, several columns added in one outer iteration, and the same growth decisions as the
    oracle in the first outer iterations."""
    rng = np.random.default_rng(60)
    edges = set()
    while len(edges) < 150:
        i, j = sorted(int(x) for x in rng.integers(0, 60, 2))
        if i != j:
            edges.add((i, j))
    P = _graph_maxcut(60, sorted(edges))
    o = oracle_mod.Oracle(P)
    R0 = inputs._unit_rows(np.random.default_rng(1), 60, 1)
    ref = alm.solve(o, R0, np.zeros(60), 1.0, alm.Params(eps=1e-7, p_max=3))
    out = gpu_solve(torch, binding, P, inputs.F64, R0, np.zeros(60), 1.0, r_cap=32, eps=1e-7, p_max=3)
    assert out["ok"] and ref.converged
    assert max(rec.grew for rec in out["log"]) >= 2
    assert abs(o.inner_C(out["R"], out["R"]) - o.inner_C(ref.R, ref.R)) <= 1e-5 * abs(o.inner_C(ref.R, ref.R))
    for a, b in list(zip(out["log"], ref.log))[:3]:
        assert (a.r, a.grew) == (b.r, b.grew), (a.t, a.r, a.grew, b.r, b.grew)
    # K_9 with p_max = 4 still reaches -n^2/4
    n = 9
    Pk = _graph_maxcut(n, [(i, j) for i in range(n) for j in range(i + 1, n)])
    outk = gpu_solve(torch, binding, Pk, inputs.F64, inputs._unit_rows(np.random.default_rng(9), n, 1), np.zeros(n), 1.0,
                     r_cap=32, eps=1e-7, p_max=4)
    assert outk["ok"] and abs(oracle_mod.Oracle(Pk).inner_C(outk["R"], outk["R"]) + n * n / 4) < 1e-4
