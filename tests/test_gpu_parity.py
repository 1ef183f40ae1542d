"""GPU parity: the CUDA path (through the C ABI) against the oracle, element by element, on the
same seeded inputs.  Tolerances (BASELINE.json north_star; definitions in DESIGN.md reading 22):
rel <= 1e-10 in fp64 and <= 2e-5 in fp32 on f, ||G||_F and z = A(RR^T); additionally on G itself,
on p0..p4 (relative to sum |p_k|) and on S(mu)v."""
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


def tdtype(torch, w):
    return torch.float32 if w.dtype == inputs.F32 else torch.float64


def dev(torch, a, dt):
    return torch.as_tensor(np.ascontiguousarray(a), dtype=dt).cuda()


def rel(a, b):
    return float(np.linalg.norm(np.asarray(a, float) - np.asarray(b, float)) / max(1e-300, np.linalg.norm(np.asarray(b, float))))


def worst_row(got, ref, extra=0.0):
    """max over rows j of ||got_j - ref_j|| / (||ref_j|| + ||ref||_F / sqrt(n) + extra_j): a single bad row (a ragged
    tail, a heavy row, a mis-staged tile) shows up here at full size, where it moves the whole-array ratio by only
    1 / sqrt(n).  The floor ||ref||_F / sqrt(n) is the typical row norm (rows that cancel are measured against it)."""
    got = np.asarray(got, float).reshape(len(ref), -1); ref = np.asarray(ref, float).reshape(len(ref), -1)
    err = np.linalg.norm(got - ref, axis=1)
    den = np.linalg.norm(ref, axis=1) + np.linalg.norm(ref) / np.sqrt(max(1, len(ref))) + extra
    j = int(np.argmax(err / np.maximum(den, 1e-300)))
    return float(err[j] / max(den[j], 1e-300)), j


def check_workload(torch, binding, oracle_mod, w, ld=None, label="", split_scale=False):
    P, tol = w.problem, TOL[w.dtype]
    o = oracle_mod.Oracle(P)
    dt = tdtype(torch, w)
    r = w.r
    ld = ld or r
    ctx = binding.Context(P, w.dtype)
    Rh = np.zeros((P.n, ld)); Rh[:, :r] = w.R
    Dh = np.zeros((P.n, ld)); Dh[:, :r] = w.D
    if ld > r:  # pads hold garbage the kernels must ignore
        Rh[:, r:] = 7.0; Dh[:, r:] = -3.0
    R, D = dev(torch, Rh, dt), dev(torch, Dh, dt)
    G = torch.full_like(R, 5.0)
    y = dev(torch, w.y, torch.float64)
    z = torch.zeros(P.m, dtype=torch.float64, device="cuda")
    ctx.set_dual(y, w.sigma)
    st = ctx.eval(R, r, ld, G, z)
    torch.cuda.synchronize()
    # oracle on the same (fp32-rounded) inputs, all arithmetic in double
    parts = o.f(w.y, w.sigma, w.R, parts=True)
    Go = o.grad(w.y, w.sigma, w.R)
    zo = o.A_op(w.R)
    fden = abs(parts["cx"]) + abs(parts["yq"]) + 0.5 * w.sigma * parts["qq"]
    assert abs(st[0] - parts["f"]) <= tol * fden, (label, st[0], parts["f"])
    assert abs(st[1] - parts["cx"]) <= tol * fden
    zg = z.cpu().numpy()
    assert rel(zg, zo) <= tol, label
    # per constraint: |dz_i| against |z_i|, the typical |z| and -- for constraints whose terms cancel -- the sum of
    # the absolute values of the terms (|A|(|R||R|^T), from the oracle run on |A|, |R|)
    zabs = oracle_mod.Oracle(_abs_problem(P)).A_op(np.abs(w.R)) if P.m else np.zeros(0)
    if P.m:
        ez, iz = worst_row(zg, zo, extra=zabs if split_scale else 0.0)
        assert ez <= tol, (label, "worst constraint", iz, ez)
    Gg = G.cpu().numpy().astype(float)
    # per row of G: the error a row inherits from lambda_i = y_i - sigma (z_i - b_i) is sigma |dz_i| <= sigma tol |z|_i
    # times the rows it multiplies ("Precision"); rowext carries that term
    lam_scale = w.sigma * tol * (zabs if split_scale else np.abs(zo))
    rowext = _adjoint_abs(P, lam_scale, np.abs(w.R)) / tol if P.m else 0.0
    if split_scale:
        # tiny degenerate problems: G = 2(CR - A*(lambda)R) may cancel almost completely (one row, one
        # constraint), so the error is measured against the two terms that are subtracted
        CR = o.smatvec(np.zeros(P.m), w.R)
        gden = 2.0 * (np.linalg.norm(CR) + np.linalg.norm(0.5 * Go - CR))
        assert np.linalg.norm(Gg[:, :r] - Go) <= tol * gden, label
        rows_split = 2.0 * (np.linalg.norm(CR, axis=1) + np.linalg.norm(0.5 * Go - CR, axis=1))
        eg, jg = worst_row(Gg[:, :r], Go, extra=rows_split + rowext)
        assert eg <= tol, (label, "worst row of G", jg, eg)
    else:
        assert rel(Gg[:, :r], Go) <= tol, label
        eg, jg = worst_row(Gg[:, :r], Go, extra=rowext)
        assert eg <= tol, (label, "worst row of G", jg, eg)
    assert abs(np.sqrt(st[4]) - np.linalg.norm(Go)) <= tol * (gden if split_scale else np.linalg.norm(Go))
    assert abs(st[5] - np.vdot(Go, w.R)) <= tol * ((gden if split_scale else np.linalg.norm(Go)) * np.linalg.norm(w.R))
    if ld > r:
        assert np.all(Gg[:, r:] == 5.0), "pad columns of G must not be touched"
    # value-only call gives the same scalars
    st2 = ctx.eval(R, r, ld, None, None)
    assert st2[0] == st[0] and st2[3] == st[3]
    # lambda
    lam = torch.zeros(P.m, dtype=torch.float64, device="cuda")
    ctx.eval(R, r, ld, G, z)
    ctx.get_lambda(lam)
    lamo, _ = o.lam(w.y, w.sigma, w.R)
    torch.cuda.synchronize()
    assert np.linalg.norm(lam.cpu().numpy() - lamo) <= tol * (np.linalg.norm(w.y) + w.sigma * np.linalg.norm(zo)), label
    # line search: cold, then warm (the ctx holds the evaluation of this same R)
    p = ctx.linesearch(R, D, r, ld)
    po = o.linesearch(w.y, w.sigma, w.R, w.D)
    assert np.abs(p - po).max() <= tol * np.abs(po).sum(), (label, p, po)
    pw = ctx.linesearch(R, D, r, ld, warm=True)
    assert np.abs(pw - po).max() <= tol * np.abs(po).sum(), (label, pw, po)
    ctx.eval(R, r, ld, None, None)                        # a value-only evaluation on record: warm without a gradient
    pw2 = ctx.linesearch(R, D, r, ld, warm=True)
    assert np.abs(pw2 - po).max() <= tol * np.abs(po).sum(), (label, pw2, po)
    ctx.eval(R, r, ld, G, z)
    with pytest.raises(binding.AloraError) as e:          # no evaluation of D on record
        ctx.linesearch(D, R, r, ld, warm=True)
    assert e.value.status == binding.ESTATE
    # matvec
    mu = dev(torch, lamo, torch.float64)
    V = dev(torch, w.V, dt)
    W = torch.zeros_like(V)
    vw = ctx.smatvec(mu, V, 1, W)
    Wo = o.smatvec(lamo, w.V)
    assert rel(W.cpu().numpy(), Wo) <= tol, label
    ew, jw = worst_row(W.cpu().numpy(), Wo, extra=_smat_abs(P, lamo, np.abs(w.V)) if split_scale else 0.0)
    assert ew <= tol, (label, "worst row of S(mu)v", jw, ew)
    assert abs(vw - w.V @ Wo) <= tol * np.linalg.norm(w.V) * np.linalg.norm(Wo)
    # mu = NULL: lambda of the last evaluation (the ctx still holds the evaluation of R above)
    W0 = torch.zeros_like(V)
    ctx.smatvec(None, V, 1, W0)
    # the library's lambda carries sigma |dz_i| <= lam_scale_i per constraint; that perturbs S(lambda) v by at most
    # sum_i lam_scale_i |A_i| |v|
    dW = 0.5 * np.linalg.norm(_adjoint_abs(P, lam_scale, np.abs(w.V).reshape(-1, 1))) if P.m else 0.0
    assert np.linalg.norm(W0.cpu().numpy().astype(float) - Wo) <= tol * np.linalg.norm(Wo) + dW, label
    # block matvec with p = 3 columns
    V3h = np.stack([w.V, np.roll(w.V, 1), w.V ** 2], axis=1)
    if w.dtype == inputs.F32:
        V3h = V3h.astype(np.float32).astype(float)
    V3 = dev(torch, V3h, dt); W3 = torch.zeros_like(V3)
    ctx.smatvec(mu, V3, 3, W3, fetch=False)
    torch.cuda.synchronize()
    assert rel(W3.cpu().numpy(), o.smatvec(lamo, V3h)) <= tol, label
    ctx.close()


def _abs_problem(P):
    """the same problem with |a_e| for every stored constraint entry (inputs for an error scale, not a result)"""
    return inputs.Problem(**{**P.__dict__, "A_val": np.abs(P.A_val), "C_val": np.abs(P.C_val),
                             "C_U": None if P.C_U is None else np.abs(P.C_U), "C_s": None if P.C_s is None else np.abs(P.C_s)})


def _adjoint_abs(P, wts, Rabs):
    """row norms of sum_i wts_i |A_i| Rabs  (scale of the error that a perturbation wts of lambda causes in G / 2)"""
    n = P.n
    out = np.zeros_like(Rabs)
    cons = np.repeat(np.arange(P.m), np.diff(P.A_ptr))
    wv = wts[cons] * np.abs(P.A_val)
    np.add.at(out, P.A_row, wv[:, None] * Rabs[P.A_col])
    off = P.A_row != P.A_col
    np.add.at(out, P.A_col[off], wv[off, None] * Rabs[P.A_row[off]])
    return 2.0 * np.linalg.norm(out, axis=1)


def _smat_abs(P, mu, Vabs):
    """row scale of S(mu) v when its terms cancel: (|C| + sum |mu_i| |A_i|) |v| (low-rank cost term included)"""
    Vabs = Vabs.reshape(P.n, -1)
    out = np.zeros_like(Vabs)
    np.add.at(out, P.C_row, np.abs(P.C_val)[:, None] * Vabs[P.C_col])
    off = P.C_row != P.C_col
    np.add.at(out, P.C_col[off], np.abs(P.C_val)[off, None] * Vabs[P.C_row[off]])
    if P.pC:
        out += np.abs(P.C_U) @ (np.abs(P.C_s)[:, None] * (np.abs(P.C_U).T @ Vabs))
    return np.linalg.norm(out, axis=1) + _adjoint_abs(P, np.abs(mu), Vabs) / 2.0


@pytest.mark.parametrize("idx", [0, 1, 2, 3, 4, 5, 6, 7])
def test_small_configs(torch, binding, oracle_mod, idx):
    check_workload(torch, binding, oracle_mod, inputs.small(idx), label=f"small{idx}")


@pytest.mark.parametrize("idx,ld", [(1, 20), (3, 12), (4, 11), (0, 41), (2, 26), (5, 4), (5, 8), (6, 20), (6, 17)])
def test_padded_leading_dimension(torch, binding, oracle_mod, idx, ld):
    """ld > r, including odd ld (element-wise path) and ld that allows wider vectors than r."""
    check_workload(torch, binding, oracle_mod, inputs.small(idx), ld=ld, label=f"small{idx}/ld{ld}")


@pytest.mark.parametrize("r", [1, 2, 3, 5, 7, 8, 13, 16, 32, 33, 64])   # 8 / 16 / 32: the dense (compile-time ld) variants incl. the bank-swizzled ones
def test_ranks(torch, binding, oracle_mod, r):
    """every (GS, NIT) shape and ragged tails, both classes and dtypes."""
    for maker in (lambda: inputs.config1(side=23, r=r), lambda: inputs.config6(side=19, r=r),
                  lambda: inputs.config3(n=700, m=900, nnzC=2000, r=r),
                  lambda: inputs.config2(n=300, M=900, r=r), lambda: inputs.config0(n=300, M=700, r=r)):
        check_workload(torch, binding, oracle_mod, maker(), label=f"r{r}")


@pytest.mark.parametrize("sel", ["0", "1"])
def test_dense_variants_both_neighbour_load_forms(torch, binding, oracle_mod, monkeypatch, sel):
    """The dense (compile-time ld) variants of the tiled kernel exist with a branch per neighbour load and with predicated
    load pairs; a call picks by the share of far neighbours, which small problems never have.  ALORA_SEL (read at
    alora_create) forces either form: both must match the oracle, on the bank-swizzled shapes (r = 16, 32 in fp32; 8, 16 in
    fp64) and a plain one, with rows that have more neighbours than ELL slots (G(n,M)) and without (torus)."""
    monkeypatch.setenv("ALORA_SEL", sel)
    for maker in (lambda: inputs.config1(side=23, r=16), lambda: inputs.config1(side=23, r=32), lambda: inputs.config1(side=23, r=8),
                  lambda: inputs.config0(n=300, M=700, r=8), lambda: inputs.config0(n=300, M=700, r=16)):
        check_workload(torch, binding, oracle_mod, maker(), label=f"sel{sel}")


@pytest.mark.parametrize("idx", [1, 2, 3, 4, 5, 6, 7])
def test_full_configs(torch, binding, oracle_mod, idx):
    """BASELINE.json's full sizes, ld = r as bench.py launches them; the C oracle is fast enough to check
    every element of z, G, S(mu)v (config 4: n = 2^24, about a minute of oracle time)."""
    check_workload(torch, binding, oracle_mod, inputs.full(idx), label=f"full{idx}")


def _edge_problems():
    from tests.helpers import problem_from_lists
    out = []
    # n = 1, one diagonal constraint, no off-diagonal cost
    out.append(("n1", problem_from_lists(1, [(0, 0, -0.5)], [[(0, 0, 1.0)]], [1.0])))
    # empty cost, constraints with zero entries (z_i = 0), duplicates, an isolated vertex (row 3)
    out.append(("empty_C", problem_from_lists(5, [], [[], [(0, 1, 0.5), (0, 1, 0.25)], [(2, 2, 1.0)], []], [0.3, 0.1, 1.0, -0.2])))
    # diagonal class with a non-identity map: constraints in reverse order, one row unconstrained, coefficients != 1
    n = 9
    C = [(j, j + 1, 1.0 + 0.1 * j) for j in range(n - 1)] + [(j, j, -0.3 * j) for j in range(n)]
    A = [[(n - 1 - i, n - 1 - i, 1.0 + 0.5 * i)] for i in range(n - 1)]
    out.append(("diag_perm", problem_from_lists(n, C, A, [1.0 + 0.1 * i for i in range(n - 1)])))
    # one long constraint (> 128 entries) next to single-entry ones, and a dense cost row (degree n-1)
    n = 300
    C = [(0, k, 0.01 * k) for k in range(1, n)]
    A = [[(j, j, 1.0) for j in range(n)] + [(j, (j + 7) % n, 0.5) if j < (j + 7) % n else ((j + 7) % n, j, 0.5) for j in range(n)]]
    A += [[(j, j + 1, 0.5)] for j in range(0, n - 1, 3)]
    out.append(("long_cons", problem_from_lists(n, C, A, [1.0] + [0.0] * (len(A) - 1))))
    return out


@pytest.mark.parametrize("dtype", [inputs.F64, inputs.F32])
@pytest.mark.parametrize("r", [1, 4, 10])
def test_edge_cases(torch, binding, oracle_mod, dtype, r):
    """degenerate inputs: n = 1, empty cost, empty constraints, duplicates, permuted / weighted diagonal
    constraints (k_rows fallback of the diagonal class), a long constraint, a dense cost row."""
    rng = np.random.default_rng(77 + r)
    for name, P in _edge_problems():
        def draw(shape):
            a = rng.standard_normal(shape)
            return a.astype(np.float32).astype(float) if dtype == inputs.F32 else a
        if dtype == inputs.F32:
            P.C_val = P.C_val.astype(np.float32).astype(float); P.A_val = P.A_val.astype(np.float32).astype(float)
        w = inputs.Workload(name=name, problem=P, dtype=dtype, r=r, R=draw((P.n, r)), y=rng.standard_normal(P.m),
                            sigma=2.5, D=draw((P.n, r)), V=draw(P.n))
        check_workload(torch, binding, oracle_mod, w, label=f"{name}/r{r}/{dtype}", split_scale=True)


def _fuzz_problem(rng, kind):
    """Random structures that walk the dispatch: `general` = random constraints (0..150 entries: short lists,
    single entries, chunked long ones), optional low-rank cost term; `diag` = one unit diagonal constraint per
    row with random row degrees around the ELL slot counts (overflow rows); `hub` = the same with one row of
    degree > 512 (general path, heavy-row segments)."""
    from tests.helpers import problem_from_lists, random_problem
    if kind == "general":
        n = int(rng.integers(2, 1500)); m = int(rng.integers(1, 2 * n))
        return random_problem(rng, n, m, max_nnz=int(rng.choice([1, 3, 8, 150])), nnzC=int(rng.integers(0, 6 * n)),
                              pC=int(rng.choice([0, 0, 1, 3])))
    n = int(rng.integers(130, 2500))
    C = {}
    for j in range(n):
        for _ in range(int(rng.integers(0, 7 if kind == "diag" else 4))):
            k = int(rng.integers(n))
            if k != j:
                C[(min(j, k), max(j, k))] = float(rng.standard_normal())
        if rng.random() < 0.3:
            C[(j, j)] = float(rng.standard_normal())
    if kind == "hub":
        h = int(rng.integers(n))
        for k in rng.choice(n, size=min(n - 1, 700), replace=False):
            if int(k) != h:
                C[(min(h, int(k)), max(h, int(k)))] = float(rng.standard_normal())
    Cl = sorted((j, k, v) for (j, k), v in C.items())
    return problem_from_lists(n, Cl, [[(j, j, 1.0)] for j in range(n)], [1.0] * n)


@pytest.mark.parametrize("seed", range(12))
def test_random_structures(torch, binding, oracle_mod, seed):
    rng = np.random.default_rng(9000 + seed)
    kind = ["general", "diag", "hub"][seed % 3]
    dtype = inputs.F32 if (seed // 3) % 2 else inputs.F64
    P = _fuzz_problem(rng, kind)
    r = int(rng.choice([1, 2, 4, 6, 10, 16, 24]))
    ld = r + int(rng.choice([0, 0, 1, 2, 4]))

    def draw(shape):
        a = rng.standard_normal(shape)
        return a.astype(np.float32).astype(float) if dtype == inputs.F32 else a
    if dtype == inputs.F32:
        P.C_val = P.C_val.astype(np.float32).astype(float); P.A_val = P.A_val.astype(np.float32).astype(float)
        if P.pC:
            P.C_U = P.C_U.astype(np.float32).astype(float)
    w = inputs.Workload(name=f"fuzz{seed}", problem=P, dtype=dtype, r=r, R=draw((P.n, r)), y=rng.standard_normal(P.m),
                        sigma=float(rng.uniform(0.1, 10.0)), D=draw((P.n, r)), V=draw(P.n))
    check_workload(torch, binding, oracle_mod, w, ld=ld, label=f"fuzz{seed}/{kind}/r{r}/ld{ld}/{dtype}", split_scale=True)


def test_m0_no_constraints(torch, binding, oracle_mod):
    """m = 0: f = <C,RR^T>, G = 2CR, S = C."""
    from tests.helpers import problem_from_lists
    P = problem_from_lists(6, [(0, 1, 1.0), (1, 2, -2.0), (3, 3, 0.7), (4, 5, 0.5)], [], [])
    rng = np.random.default_rng(5)
    w = inputs.Workload(name="m0", problem=P, dtype=inputs.F64, r=3, R=rng.standard_normal((6, 3)), y=np.zeros(0),
                        sigma=1.0, D=rng.standard_normal((6, 3)), V=rng.standard_normal(6))
    check_workload(torch, binding, oracle_mod, w, label="m0")


def test_cuda_graph_capture_of_a_step(torch, binding, oracle_mod):
    """The three hot-path calls enqueue kernels only (no synchronisation, no allocation) when no host output is
    requested, so a step can be captured into a CUDA graph on the ctx stream and replayed; the replay gives the
    same scalars and arrays as the direct calls."""
    w = inputs.small(1)
    P, r = w.problem, w.r
    s = torch.cuda.Stream()
    s.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(s):
        ctx = binding.Context(P, w.dtype, stream=s.cuda_stream)
        R = dev(torch, w.R, torch.float32); D = dev(torch, w.D, torch.float32); V = dev(torch, w.V, torch.float32)
        G = torch.zeros_like(R); W = torch.zeros_like(V)
        y = dev(torch, w.y, torch.float64)
        z = torch.zeros(P.m, dtype=torch.float64, device="cuda"); lam = torch.zeros_like(z)
        ctx.set_dual(y, w.sigma)
        st0 = ctx.eval(R, r, r, G, z); ctx.get_lambda(lam)
        p0 = ctx.linesearch(R, D, r, r)
        ctx.smatvec(lam, V, 1, W, fetch=False)
        torch.cuda.synchronize()
        G0, W0 = G.clone(), W.clone()
        G.zero_(); W.zero_()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=s):
            ctx.eval(R, r, r, G, z, stats=False)
            ctx.linesearch(R, D, r, r, fetch=False)
            ctx.smatvec(lam, V, 1, W, fetch=False)
        G.zero_(); W.zero_()
        g.replay(); g.replay()
        torch.cuda.synchronize()
        assert torch.equal(G, G0) and torch.equal(W, W0)
        assert np.array_equal(ctx.get_stats(), st0) and np.array_equal(ctx.get_linesearch(), p0)
        ctx.close()
