"""Seeded synthetic input generators (shared by the oracle tests and the CUDA path).

This module only *constructs problem data*: graphs, the MaxCut cost C = -L/4 built from the
Laplacian formula (section 6.1), constraint patterns, right-hand sides and random
starting points.  It holds none of the solver's arithmetic (no f, no gradient, no line search, no
matvec, no random numbers the method draws) and imports neither ``oracle/`` nor the CUDA binding.
Both sides consume the arrays it returns.  One piece of data construction restates a definition of the
paper: ``planted_rhs`` forms b_i = <A_i, R0 R0^T> for BASELINE.json's config 3 with numpy,
because b IS the workload there; it feeds neither side's results, and tests/test_inputs.py and
tests/test_oracle_pins.py check it against the oracle's own A(.).

Storage convention: **sym-upper COO** -- an entry ``(j, k, a)`` with
``j <= k`` means ``A[j,k] = A[k,j] = a``.  Constraints are stacked: entries
``A_ptr[i]:A_ptr[i+1]`` belong to ``A_i`` (section 1.2).

The paper's own workloads are DIMACS10 graphs which are not available offline; the
recipes below (BASELINE.json configs 0-4) stand in for them.
Every generator is driven by ``numpy.random.Generator(PCG64(seed))`` with
``seed = 1000 + config index``.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Optional

import numpy as np

F32 = "f32"
F64 = "f64"


@dataclass
class Problem:
    """SDP data  min <C,X>  s.t.  <A_i,X> = b_i,  X psd   (problem (P))."""

    n: int
    m: int
    C_row: np.ndarray  # int32 [nnzC], row <= col
    C_col: np.ndarray  # int32 [nnzC]
    C_val: np.ndarray  # float64 [nnzC]
    A_ptr: np.ndarray  # int64 [m+1]
    A_row: np.ndarray  # int32 [nnzA], row <= col
    A_col: np.ndarray  # int32 [nnzA]
    A_val: np.ndarray  # float64 [nnzA]
    b: np.ndarray  # float64 [m]
    # optional low-rank cost term  C += U diag(s) U^T,  U is n x pC (column-major when flattened)
    C_U: Optional[np.ndarray] = None  # float64 [n, pC]
    C_s: Optional[np.ndarray] = None  # float64 [pC]

    @property
    def pC(self) -> int:
        return 0 if self.C_s is None else int(self.C_s.shape[0])

    @property
    def nnzC(self) -> int:
        return int(self.C_val.shape[0])

    @property
    def nnzA(self) -> int:
        return int(self.A_val.shape[0])


@dataclass
class Workload:
    """A problem plus the point at which the hot path is evaluated."""

    name: str
    problem: Problem
    dtype: str  # F32 or F64: storage type of R / D / G and of the stored values
    r: int
    R: np.ndarray  # float64 [n, r] (fp32-representable when dtype == F32)
    y: np.ndarray  # float64 [m]
    sigma: float
    D: np.ndarray  # float64 [n, r] search direction for the line-search coefficients
    V: np.ndarray  # float64 [n]    test vector for the Lanczos matvec
    meta: dict = field(default_factory=dict)


def _rng(seed: int) -> np.random.Generator:
    return np.random.Generator(np.random.PCG64(seed))


def _round_f32(x: np.ndarray) -> np.ndarray:
    """Round to the nearest fp32 value, returned widened back to float64."""
    return np.asarray(x, dtype=np.float32).astype(np.float64)


def _unit_rows(rng: np.random.Generator, n: int, r: int) -> np.ndarray:
    """R ~ N(0,1) i.i.d., then each row scaled to unit Euclidean norm (BASELINE.json config 0)."""
    R = rng.standard_normal((n, r))
    R /= np.sqrt((R * R).sum(axis=1, keepdims=True))
    return R


# ----------------------------------------------------------------------------------------------
# graphs (edge lists with i < j)
# ----------------------------------------------------------------------------------------------
def gnm_edges(rng: np.random.Generator, n: int, M: int) -> tuple[np.ndarray, np.ndarray]:
    """G(n,M): M distinct pairs i<j drawn without replacement from the n(n-1)/2 pairs."""
    total = n * (n - 1) // 2
    if M > total:
        raise ValueError("too many edges")
    if total <= 50_000_000:
        code = rng.choice(total, size=M, replace=False)
    else:  # rejection on a sparse draw
        code = np.unique(rng.integers(0, total, size=int(M * 1.1) + 16))
        rng.shuffle(code)
        if code.shape[0] < M:
            raise RuntimeError("resample")
        code = code[:M]
    code = np.sort(code.astype(np.int64))
    # decode: pairs enumerated row by row, row i holds (n-1-i) pairs
    # start(i) = i*n - i*(i+1)/2 ; invert with a float guess then fix up
    i = np.floor(((2 * n - 1) - np.sqrt((2 * n - 1) ** 2 - 8.0 * code)) / 2).astype(np.int64)
    start = i * n - i * (i + 1) // 2
    i = np.where(start > code, i - 1, i)
    start = i * n - i * (i + 1) // 2
    nxt = (i + 1) * n - (i + 1) * (i + 2) // 2
    i = np.where(code >= nxt, i + 1, i)
    start = i * n - i * (i + 1) // 2
    j = code - start + i + 1
    assert np.all((0 <= i) & (i < j) & (j < n))
    return i.astype(np.int64), j.astype(np.int64)


def torus_edges(side: int) -> tuple[np.ndarray, np.ndarray]:
    """side x side torus: vertex (a,c) -> side*a+c, edges to ((a+1) mod side, c), (a,(c+1) mod side)."""
    a, c = np.meshgrid(np.arange(side), np.arange(side), indexing="ij")
    v = (side * a + c).ravel()
    down = (side * ((a + 1) % side) + c).ravel()
    right = (side * a + (c + 1) % side).ravel()
    u = np.concatenate([v, v])
    w = np.concatenate([down, right])
    lo, hi = np.minimum(u, w), np.maximum(u, w)
    return lo.astype(np.int64), hi.astype(np.int64)


def tri_torus_edges(side: int) -> tuple[np.ndarray, np.ndarray]:
    """Triangulated side x side torus (degree 6): the torus edges plus the diagonal (a,c)-((a+1),(c+1)).
    Stand-in for the mesh / Delaunay graphs of the paper's Table 1, whose vertices have
    about six neighbours."""
    a, c = np.meshgrid(np.arange(side), np.arange(side), indexing="ij")
    v = (side * a + c).ravel()
    down = (side * ((a + 1) % side) + c).ravel()
    right = (side * a + (c + 1) % side).ravel()
    diag = (side * ((a + 1) % side) + (c + 1) % side).ravel()
    u = np.concatenate([v, v, v])
    w = np.concatenate([down, right, diag])
    lo, hi = np.minimum(u, w), np.maximum(u, w)
    return lo.astype(np.int64), hi.astype(np.int64)


def rmat_edges(rng: np.random.Generator, scale: int, edge_factor: int) -> tuple[np.ndarray, np.ndarray]:
    """R-MAT / Kronecker generator (Graph500 parameters a, b, c = 0.57, 0.19, 0.19): 2^scale vertices,
    edge_factor * 2^scale sampled edges; power-law degrees with a few very heavy rows.  Stand-in for the
    kron_g500 graphs, the slowest instances of the paper's Table 1."""
    ne = edge_factor << scale
    u = np.zeros(ne, np.int64)
    w = np.zeros(ne, np.int64)
    ab, c_norm, a_norm = 0.57 + 0.19, 0.19 / (1.0 - 0.76), 0.57 / 0.76
    for bit in range(scale):
        ii = rng.random(ne) > ab
        jj = rng.random(ne) > np.where(ii, c_norm, a_norm)
        u |= ii.astype(np.int64) << bit
        w |= jj.astype(np.int64) << bit
    return np.minimum(u, w), np.maximum(u, w)


def ring_matching_edges(rng: np.random.Generator, n: int) -> tuple[np.ndarray, np.ndarray]:
    """Ring i-(i+1) mod n plus two independent seeded random perfect matchings (n even)."""
    if n % 2:
        raise ValueError("n must be even")
    i = np.arange(n, dtype=np.int64)
    us, ws = [i], [(i + 1) % n]
    for _ in range(2):
        pi = rng.permutation(n).astype(np.int64)
        us.append(pi[0::2])
        ws.append(pi[1::2])
    u, w = np.concatenate(us), np.concatenate(ws)
    return np.minimum(u, w), np.maximum(u, w)


def coalesce_edges(lo: np.ndarray, hi: np.ndarray, w: np.ndarray, n: int):
    """Sum the weights of coincident edges, drop zero-sum edges and self loops; sort by (lo,hi)."""
    keep = lo != hi
    lo, hi, w = lo[keep], hi[keep], w[keep]
    key = lo * np.int64(n) + hi
    order = np.argsort(key, kind="stable")
    key, w = key[order], w[order]
    uniq, first = np.unique(key, return_index=True)
    wsum = np.add.reduceat(w, first) if key.size else w
    nz = wsum != 0
    uniq, wsum = uniq[nz], wsum[nz]
    return (uniq // n).astype(np.int64), (uniq % n).astype(np.int64), wsum


# ----------------------------------------------------------------------------------------------
# problem builders
# ----------------------------------------------------------------------------------------------
def maxcut_problem(n: int, lo: np.ndarray, hi: np.ndarray, w: np.ndarray) -> Problem:
    """MaxCut SDP  min <C,X>, C = -L/4, X_ii = 1  (section 6.1).

    L_ij = -w_ij on edges, L_ii = sum_k w_ik (used verbatim with signed weights),
    A_i = e_i e_i^T, b = 1.
    """
    deg = np.zeros(n)
    np.add.at(deg, lo, w)
    np.add.at(deg, hi, w)
    rows = np.concatenate([np.arange(n, dtype=np.int64), lo])
    cols = np.concatenate([np.arange(n, dtype=np.int64), hi])
    vals = np.concatenate([-deg / 4.0, w / 4.0])  # C = -L/4: diag -deg/4, off-diag +w/4
    order = np.lexsort((cols, rows))
    idx = np.arange(n, dtype=np.int32)
    return Problem(
        n=n, m=n,
        C_row=rows[order].astype(np.int32), C_col=cols[order].astype(np.int32), C_val=vals[order],
        A_ptr=np.arange(n + 1, dtype=np.int64), A_row=idx.copy(), A_col=idx.copy(),
        A_val=np.ones(n), b=np.ones(n),
    )


def theta_problem(n: int, lo: np.ndarray, hi: np.ndarray) -> Problem:
    """Lovasz theta SDP  min <-J,X>  s.t. tr X = 1, X_ij = 0 on edges (BASELINE.json config 2).

    Constraint 0 is the trace (n diagonal entries, a=1, b=1); constraint 1+e is the edge e stored
    as (i,j,1/2), i.e. A = (e_i e_j^T + e_j e_i^T)/2 as in PAPER.md:533 / :824.  The cost -J is the
    rank-one term U = 1, s = -1 (no sparse part).
    """
    M = lo.shape[0]
    d = np.arange(n, dtype=np.int32)
    return Problem(
        n=n, m=M + 1,
        C_row=np.zeros(0, np.int32), C_col=np.zeros(0, np.int32), C_val=np.zeros(0),
        A_ptr=np.concatenate([[0], n + np.arange(M + 1, dtype=np.int64)]).astype(np.int64),
        A_row=np.concatenate([d, lo.astype(np.int32)]), A_col=np.concatenate([d, hi.astype(np.int32)]),
        A_val=np.concatenate([np.ones(n), np.full(M, 0.5)]),
        b=np.concatenate([[1.0], np.zeros(M)]),
        C_U=np.ones((n, 1)), C_s=np.array([-1.0]),
    )


def _random_sym_entries(rng, n: int, count: int):
    j = rng.integers(0, n, size=count)
    k = rng.integers(0, n, size=count)
    return np.minimum(j, k).astype(np.int32), np.maximum(j, k).astype(np.int32), rng.standard_normal(count)


def planted_rhs(p_ptr, row, col, val, R0) -> np.ndarray:
    """Right-hand side of the planted instance, b_i = <A_i, R0 R0^T>  (BASELINE.json config 3).

    Data construction (fp64, numpy): diagonal entries count once, off-diagonal stored entries twice.  This is the
    one place where the generator restates a formula of the method (module docstring); it is checked against the
    oracle's A(.) in tests/test_inputs.py, and neither the oracle nor the CUDA path calls it.
    """
    w = np.where(row == col, 1.0, 2.0) * val * np.einsum("ec,ec->e", R0[row], R0[col])
    cons = np.repeat(np.arange(p_ptr.shape[0] - 1), np.diff(p_ptr))
    return np.bincount(cons, weights=w, minlength=p_ptr.shape[0] - 1)


def random_sparse_problem(rng, n: int, m: int, nnz_per_cons: int, nnzC: int, r0: int, f32: bool):
    """Random sparse-constraint SDP (BASELINE.json config 3): each A_i has `nnz_per_cons` stored
    sym-upper entries at uniform (j,k) with N(0,1) values; C likewise with nnzC entries;
    b = A(R0 R0^T) for a planted R0 ~ N(0,1/n) in R^{n x r0}."""
    ar, ac, av = _random_sym_entries(rng, n, m * nnz_per_cons)
    cr, cc, cv = _random_sym_entries(rng, n, nnzC)
    order = np.lexsort((cc, cr))
    cr, cc, cv = cr[order], cc[order], cv[order]
    if f32:
        av, cv = _round_f32(av), _round_f32(cv)
    A_ptr = np.arange(m + 1, dtype=np.int64) * nnz_per_cons
    R0 = rng.standard_normal((n, r0)) / np.sqrt(n)
    b = planted_rhs(A_ptr, ar, ac, av, R0)
    return Problem(n=n, m=m, C_row=cr, C_col=cc, C_val=cv, A_ptr=A_ptr, A_row=ar, A_col=ac,
                   A_val=av, b=b), R0


# ----------------------------------------------------------------------------------------------
# workloads: BASELINE.json configs 0..4 (full size) and scaled-down versions for parity tests
# ----------------------------------------------------------------------------------------------
def _finish(name, prob, dtype, r, R, y, sigma, rng, meta=None) -> Workload:
    n = prob.n
    D = rng.standard_normal((n, r)) * (np.abs(R).mean() if R.size else 1.0)
    V = rng.standard_normal(n)
    if dtype == F32:
        R, D, V = _round_f32(R), _round_f32(D), _round_f32(V)
    return Workload(name=name, problem=prob, dtype=dtype, r=r, R=R, y=np.asarray(y, float),
                    sigma=float(sigma), D=D, V=V, meta=meta or {})


def config0(n: int = 800, M: int = 2400, r: int = 40, seed: int = 1000) -> Workload:
    """MaxCut on G(n,M), weights +1, fp64, rows of R normalised, y = 0, sigma = 1."""
    rng = _rng(seed)
    lo, hi = gnm_edges(rng, n, M)
    prob = maxcut_problem(n, lo, hi, np.ones(M))
    R = _unit_rows(rng, n, r)
    return _finish("cfg0_maxcut_gnm", prob, F64, r, R, np.zeros(n), 1.0, rng, {"edges": M})


def config1(side: int = 1000, r: int = 16, seed: int = 1001) -> Workload:
    """MaxCut on the side x side torus, weights uniform +-1, fp32 R, y ~ N(0,1), sigma = 10."""
    rng = _rng(seed)
    lo, hi = torus_edges(side)
    w = rng.choice(np.array([-1.0, 1.0]), size=lo.shape[0])
    lo, hi, w = coalesce_edges(lo, hi, w, side * side)  # side<=2 would create duplicates
    n = side * side
    prob = maxcut_problem(n, lo, hi, w)
    R = _unit_rows(rng, n, r)
    y = rng.standard_normal(n)
    return _finish("cfg1_maxcut_torus", prob, F32, r, R, y, 10.0, rng, {"edges": int(lo.shape[0])})


def config2(n: int = 20000, M: int = 200000, r: int = 24, seed: int = 1002) -> Workload:
    """Lovasz theta on G(n,M), fp64; R ~ N(0,1/(n r)) so tr(RR^T) ~ 1, y ~ N(0,1), sigma = 1."""
    rng = _rng(seed)
    lo, hi = gnm_edges(rng, n, M)
    prob = theta_problem(n, lo, hi)
    R = rng.standard_normal((n, r)) / np.sqrt(n * r)
    y = rng.standard_normal(prob.m)
    return _finish("cfg2_theta_gnm", prob, F64, r, R, y, 1.0, rng, {"edges": M})


def config3(n: int = 100000, m: int = 500000, nnzC: int = 1000000, r: int = 10,
            seed: int = 1003) -> Workload:
    """Random sparse-constraint SDP, fp32 values / fp64 sums; R ~ N(0,1/n), y ~ N(0,1), sigma = 10."""
    rng = _rng(seed)
    prob, R0 = random_sparse_problem(rng, n, m, 4, nnzC, 5, f32=True)
    R = rng.standard_normal((n, r)) / np.sqrt(n)
    y = rng.standard_normal(m)
    return _finish("cfg3_random_sparse", prob, F32, r, R, y, 10.0, rng, {"planted_rank": 5})


def config4(n: int = 1 << 24, r: int = 10, seed: int = 1004) -> Workload:
    """Large MaxCut: ring + two random perfect matchings, weights +-1, fp32 R, y = 0, sigma = 1."""
    rng = _rng(seed)
    lo, hi = ring_matching_edges(rng, n)
    w = rng.choice(np.array([-1.0, 1.0]), size=lo.shape[0])
    lo, hi, w = coalesce_edges(lo, hi, w, n)
    prob = maxcut_problem(n, lo, hi, w)
    R = _unit_rows(rng, n, r)
    return _finish("cfg4_maxcut_ring_matchings", prob, F32, r, R, np.zeros(n), 1.0, rng,
                   {"edges": int(lo.shape[0])})


def matrix_completion_problem(rng, n1: int, n2: int, r_star: int, m: int):
    """Matrix-completion SDP of PAPER.md:997-1008 (section 6.2):  min 1/2 tr X  s.t.
    X = [[W1, Y], [Y^T, W2]] psd,  Y_ij = M_ij on Omega,  with M = U V^T, U (n1 x r*) and V (n2 x r*)
    standard Gaussian and |Omega| = m entries drawn uniformly without replacement.

    Constraint for (i, j) in Omega: X[i, n1 + j] = M_ij, i.e. A = (e_i e_k^T + e_k e_i^T)/2 with
    k = n1 + j, stored sym-upper as (i, k, 1/2)  (PAPER.md:533 convention); cost C = I/2.
    Returns (Problem, U, V)."""
    n = n1 + n2
    if m > n1 * n2:
        raise ValueError("more observations than entries")
    U, V = rng.standard_normal((n1, r_star)), rng.standard_normal((n2, r_star))
    # m distinct flat positions in [0, n1*n2): draw with replacement, drop duplicates, top up
    flat = np.unique(rng.integers(0, n1 * n2, size=m, dtype=np.int64))
    while flat.shape[0] < m:
        extra = rng.integers(0, n1 * n2, size=m - flat.shape[0], dtype=np.int64)
        flat = np.unique(np.concatenate([flat, extra]))
    i, j = (flat // n2).astype(np.int32), (flat % n2).astype(np.int32)
    b = np.einsum("ec,ec->e", U[i], V[j])
    d = np.arange(n, dtype=np.int32)
    prob = Problem(n=n, m=m, C_row=d, C_col=d.copy(), C_val=np.full(n, 0.5),
                   A_ptr=np.arange(m + 1, dtype=np.int64), A_row=i, A_col=(n1 + j).astype(np.int32),
                   A_val=np.full(m, 0.5), b=b)
    return prob, U, V


def mc_observations(n: int, r_star: int) -> int:
    """m = ceil(gamma r* (n - r*)), gamma = r* log n."""
    return int(np.ceil(r_star * np.log(n) * r_star * (n - r_star)))


def config5(n: int = 10000, r_star: int = 3, r: int = 0, seed: int = 1005, m: int = 0) -> Workload:
    """Matrix completion (first row of the paper's Table 2 by default: r* = 3,
    n = 10000, m = 828659), n1 = n2 = n/2, fp32 R / fp64 sums.  The paper is silent on R0, y0, sigma:
    R ~ N(0,1) (the scale of the factors of M), y = 0, sigma = 1; the BM rank defaults to r*."""
    rng = _rng(seed)
    n1 = n // 2
    m = m or mc_observations(n, r_star)
    prob, U, V = matrix_completion_problem(rng, n1, n - n1, r_star, m)
    r = r or r_star
    R = rng.standard_normal((n, r))
    y = np.zeros(m) if m > 4000000 else rng.standard_normal(m) * 0.1
    return _finish("cfg5_matrix_completion", prob, F32, r, R, y, 1.0, rng,
                   {"r_star": r_star, "n1": n1, "n2": n - n1, "U": U, "V": V})


def config6(side: int = 1000, r: int = 16, seed: int = 1006) -> Workload:
    """MaxCut on the triangulated torus (degree 6, mesh stand-in), unit weights as in the paper's MaxCut runs
    (PAPER.md:969), fp32 R, y ~ N(0,1), sigma = 10.  Exercises the wide ELL variant of the tiled kernel."""
    rng = _rng(seed)
    lo, hi = tri_torus_edges(side)
    lo, hi, w = coalesce_edges(lo, hi, np.ones(lo.shape[0]), side * side)
    n = side * side
    prob = maxcut_problem(n, lo, hi, w)
    R = _unit_rows(rng, n, r)
    y = rng.standard_normal(n)
    return _finish("cfg6_maxcut_tri_torus", prob, F32, r, R, y, 10.0, rng, {"edges": int(lo.shape[0])})


def config7(scale: int = 20, edge_factor: int = 8, r: int = 16, seed: int = 1007) -> Workload:
    """MaxCut on an R-MAT graph (load-balance stress): unit weights, fp32 R."""
    rng = _rng(seed)
    lo, hi = rmat_edges(rng, scale, edge_factor)
    n = 1 << scale
    lo, hi, w = coalesce_edges(lo, hi, np.ones(lo.shape[0]), n)
    w = np.ones_like(w)   # simple graph: repeated samples of an edge count once
    prob = maxcut_problem(n, lo, hi, w)
    R = _unit_rows(rng, n, r)
    y = rng.standard_normal(n)
    return _finish("cfg7_maxcut_rmat", prob, F32, r, R, y, 10.0, rng, {"edges": int(lo.shape[0])})


CONFIGS = [config0, config1, config2, config3, config4, config5, config6, config7]

# scaled-down versions: several tiles plus a ragged tail, oracle finishes in well under a second
SMALL = {
    0: lambda: config0(n=800, M=2400, r=40),
    1: lambda: config1(side=37, r=16),
    2: lambda: config2(n=701, M=5003, r=24),
    3: lambda: config3(n=3001, m=15007, nnzC=30011, r=10),
    4: lambda: config4(n=20002, r=10),
    5: lambda: config5(n=601, r_star=3, r=4, m=20011),
    6: lambda: config6(side=41, r=16),
    7: lambda: config7(scale=11, edge_factor=8, r=16),
}


def small(idx: int) -> Workload:
    return SMALL[idx]()


def full(idx: int) -> Workload:
    return CONFIGS[idx]()
