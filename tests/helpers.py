"""Test helpers: tiny problems from explicit entry lists, dense brute-force formulas (numpy)."""
import numpy as np

from paper_2505_15775_b200.inputs import Problem


def problem_from_lists(n, C, A, b, U=None, s=None):
    """C: [(j,k,v)] sym-upper; A: list (one per constraint) of [(j,k,v)] sym-upper."""
    ptr, ar, ac, av = [0], [], [], []
    for Ai in A:
        for (j, k, v) in Ai:
            assert j <= k
            ar.append(j); ac.append(k); av.append(v)
        ptr.append(len(ar))
    return Problem(
        n=n, m=len(A),
        C_row=np.array([e[0] for e in C], np.int32), C_col=np.array([e[1] for e in C], np.int32),
        C_val=np.array([e[2] for e in C], float),
        A_ptr=np.array(ptr, np.int64), A_row=np.array(ar, np.int32), A_col=np.array(ac, np.int32),
        A_val=np.array(av, float), b=np.array(b, float),
        C_U=None if U is None else np.asarray(U, float), C_s=None if s is None else np.asarray(s, float))


def dense_matrices(P):
    """Dense C (with low-rank term) and the list of dense A_i from the sym-upper COO."""
    n = P.n
    Cd = np.zeros((n, n))
    for j, k, v in zip(P.C_row, P.C_col, P.C_val):
        Cd[j, k] += v
        if j != k:
            Cd[k, j] += v
    if P.pC:
        Cd += P.C_U @ np.diag(P.C_s) @ P.C_U.T
    Ad = []
    for i in range(P.m):
        M = np.zeros((n, n))
        for e in range(P.A_ptr[i], P.A_ptr[i + 1]):
            j, k, v = P.A_row[e], P.A_col[e], P.A_val[e]
            M[j, k] += v
            if j != k:
                M[k, j] += v
        Ad.append(M)
    return Cd, Ad


def random_problem(rng, n, m, max_nnz=5, nnzC=None, pC=0, diag_frac=0.3):
    """Random sparse symmetric data with a mix of diagonal / off-diagonal entries, duplicate
    entries inside a constraint allowed (they must be summed)."""
    def entries(cnt):
        out = []
        for _ in range(cnt):
            if rng.random() < diag_frac:
                j = k = int(rng.integers(n))
            else:
                j, k = sorted(int(x) for x in rng.integers(n, size=2))
            out.append((j, k, float(rng.standard_normal())))
        return out
    A = [entries(int(rng.integers(0, max_nnz + 1))) for _ in range(m)]
    C = entries(nnzC if nnzC is not None else 2 * n)
    C.sort()
    U = rng.standard_normal((n, pC)) if pC else None
    s = rng.standard_normal(pC) if pC else None
    return problem_from_lists(n, C, A, rng.standard_normal(m), U, s)
