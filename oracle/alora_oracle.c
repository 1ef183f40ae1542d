/*
 * alora_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, obviously-correct CPU implementation (fp64, single thread, straight loops over
 * the stored entries) of what the ALM-BM hot path of ALORA (arXiv 2505.15775) computes.
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * call it.  It shares no code with the CUDA path (paper_2505_15775_b200/csrc) and includes none
 * of its headers.
 *
 * Every function is the paper's definition written out:
 *   (P)      min <C,X>  s.t.  [A(X)]_i = <A_i,X> = b_i,  X psd           PAPER.md:85-91  (sec 1.2)
 *   (AL-BM)  f(R) = <C,RR^T> + <y, b - A(RR^T)> + (sigma/2)||A(RR^T)-b||^2
 *   grad     nabla f(R) = 2 [C - A^*(y + sigma(b - A(RR^T)))] R
 *   Z(y)     = C - A^*(y),  A^*(w) = sum_i w_i A_i
 * (paper's F, rho, L-bar are R, sigma, f here -- BASELINE.json's notation).
 *
 * Storage: sym-upper COO.  A stored entry (j,k,a) with j<=k means A[j,k]=A[k,j]=a, so in a trace
 * inner product <A,M> with M symmetric it counts once if j==k and twice if j<k.  This matches the
 * paper's own examples, where "X_ij = const" is A = (e_i e_j^T + e_j e_i^T)/2.
 * Optional low-rank cost term: C_total = C + U diag(s) U^T, U is n x pC, column-major.
 *
 * Pins (tests/test_oracle_pins.py): dense X=RR^T brute force, central finite differences, the
 * quartic identity, paper eq. 36 / 42-43 / Prop. 6 / Prop. 7 values, dense eigen-solver.
 */
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

typedef struct {
  int64_t n, m;
  int64_t nnzC;
  const int32_t *C_row, *C_col;
  const double *C_val;
  int32_t pC;
  const double *C_U; /* n x pC column-major */
  const double *C_s; /* pC */
  int64_t nnzA;
  const int64_t *A_ptr; /* m+1 */
  const int32_t *A_row, *A_col;
  const double *A_val;
  const double *b; /* m */
} oracle_problem;

static double rowdot(const double *X, const double *Y, int64_t j, int64_t k, int32_t r) {
  double s = 0.0;
  for (int32_t c = 0; c < r; ++c) s += X[j * r + c] * Y[k * r + c];
  return s;
}

/* out_i = <A_i, X Y^T + Y X^T> / 2  =  sum_e  a_e * ( j==k ? <X_j,Y_j> : <X_j,Y_k> + <X_k,Y_j> ).
 * With X == Y this is [A(XX^T)]_i.  X, Y are n x r row-major. */
void oracle_A_sym(const oracle_problem *P, const double *X, const double *Y, int32_t r, double *out) {
  for (int64_t i = 0; i < P->m; ++i) {
    double s = 0.0;
    for (int64_t e = P->A_ptr[i]; e < P->A_ptr[i + 1]; ++e) {
      int64_t j = P->A_row[e], k = P->A_col[e];
      double a = P->A_val[e];
      if (j == k) s += a * rowdot(X, Y, j, j, r);
      else s += a * (rowdot(X, Y, j, k, r) + rowdot(X, Y, k, j, r));
    }
    out[i] = s;
  }
}

/* z = A(RR^T) */
void oracle_A_op(const oracle_problem *P, const double *R, int32_t r, double *z) {
  oracle_A_sym(P, R, R, r, z);
}

/* <C_total, X Y^T> for symmetric C_total (sparse part + U diag(s) U^T). */
double oracle_inner_C(const oracle_problem *P, const double *X, const double *Y, int32_t r) {
  double s = 0.0;
  for (int64_t e = 0; e < P->nnzC; ++e) {
    int64_t j = P->C_row[e], k = P->C_col[e];
    double c = P->C_val[e];
    if (j == k) s += c * rowdot(X, Y, j, j, r);
    else s += c * (rowdot(X, Y, j, k, r) + rowdot(X, Y, k, j, r));
  }
  /* <U diag(s) U^T, X Y^T> = sum_p s_p <U_p^T X, U_p^T Y> */
  for (int32_t p = 0; p < P->pC; ++p) {
    const double *u = P->C_U + (int64_t)p * P->n;
    for (int32_t c = 0; c < r; ++c) {
      double tx = 0.0, ty = 0.0;
      for (int64_t j = 0; j < P->n; ++j) { tx += u[j] * X[j * r + c]; ty += u[j] * Y[j * r + c]; }
      s += P->C_s[p] * tx * ty;
    }
  }
  return s;
}

/* f(R) = <C,RR^T> - y^T(A(RR^T)-b) + (sigma/2)||A(RR^T)-b||^2   (AL-BM; sign of y as
 * in PAPER.md:93: <y, b - AX> = -y^T(AX-b)).  parts[0..3] = <C,X>, y.q, ||q||^2, f  (may be NULL). */
double oracle_f(const oracle_problem *P, const double *y, double sigma, const double *R, int32_t r,
                double *parts) {
  double *z = (double *)malloc(sizeof(double) * (size_t)(P->m > 0 ? P->m : 1));
  oracle_A_op(P, R, r, z);
  double cx = oracle_inner_C(P, R, R, r), yq = 0.0, qq = 0.0;
  for (int64_t i = 0; i < P->m; ++i) {
    double q = z[i] - P->b[i];
    yq += y[i] * q;
    qq += q * q;
  }
  free(z);
  double f = cx - yq + 0.5 * sigma * qq;
  if (parts) { parts[0] = cx; parts[1] = yq; parts[2] = qq; parts[3] = f; }
  return f;
}

/* W = (C_total - sum_i w_i A_i) V  for V, W n x p row-major: the dual slack map Z(w) = C - A^*(w)
 * applied to p columns.  Used for the gradient (w = lambda, V = R) and for
 * the Lanczos operator (Alg. 1 line 5; eq. 77). */
void oracle_smatvec(const oracle_problem *P, const double *w, const double *V, int32_t p, double *W) {
  memset(W, 0, sizeof(double) * (size_t)P->n * (size_t)p);
  for (int64_t e = 0; e < P->nnzC; ++e) {
    int64_t j = P->C_row[e], k = P->C_col[e];
    double c = P->C_val[e];
    for (int32_t t = 0; t < p; ++t) W[j * p + t] += c * V[k * p + t];
    if (j != k) for (int32_t t = 0; t < p; ++t) W[k * p + t] += c * V[j * p + t];
  }
  for (int32_t q = 0; q < P->pC; ++q) {
    const double *u = P->C_U + (int64_t)q * P->n;
    for (int32_t t = 0; t < p; ++t) {
      double ut = 0.0;
      for (int64_t j = 0; j < P->n; ++j) ut += u[j] * V[j * p + t];
      for (int64_t j = 0; j < P->n; ++j) W[j * p + t] += P->C_s[q] * u[j] * ut;
    }
  }
  for (int64_t i = 0; i < P->m; ++i) {
    for (int64_t e = P->A_ptr[i]; e < P->A_ptr[i + 1]; ++e) {
      int64_t j = P->A_row[e], k = P->A_col[e];
      double a = w[i] * P->A_val[e];
      for (int32_t t = 0; t < p; ++t) W[j * p + t] -= a * V[k * p + t];
      if (j != k) for (int32_t t = 0; t < p; ++t) W[k * p + t] -= a * V[j * p + t];
    }
  }
}

/* lambda = y - sigma (A(RR^T) - b)   (z_{y,rho} of PAPER.md:483 with X = RR^T);  z may be NULL */
void oracle_lambda(const oracle_problem *P, const double *y, double sigma, const double *R, int32_t r,
                   double *lambda, double *z) {
  double *zz = z ? z : (double *)malloc(sizeof(double) * (size_t)(P->m > 0 ? P->m : 1));
  oracle_A_op(P, R, r, zz);
  for (int64_t i = 0; i < P->m; ++i) lambda[i] = y[i] - sigma * (zz[i] - P->b[i]);
  if (!z) free(zz);
}

/* G = nabla f(R) = 2 (C - A^*(lambda)) R   ("nabla h(F) = 2 nabla f(X) F" with
 * nabla_X L_rho = C - A^*(y + rho(b - AX)), PAPER.md:483 / eq. 67 at :839).  Factor 2 kept
 * (reading 2; checked by finite differences in the pins). */
void oracle_grad(const oracle_problem *P, const double *y, double sigma, const double *R, int32_t r,
                 double *G) {
  double *lambda = (double *)malloc(sizeof(double) * (size_t)(P->m > 0 ? P->m : 1));
  oracle_lambda(P, y, sigma, R, r, lambda, NULL);
  oracle_smatvec(P, lambda, R, r, G);
  for (int64_t t = 0; t < P->n * (int64_t)r; ++t) G[t] *= 2.0;
  free(lambda);
}

/* Coefficients of phi(alpha) = f(R + alpha D) = sum_k p_k alpha^k.  Expanding
 * (R+aD)(R+aD)^T = RR^T + a (RD^T+DR^T) + a^2 DD^T in (AL-BM) with
 * q = A(RR^T)-b, q1 = A(RD^T+DR^T), q2 = A(DD^T):
 *   p0 = <C,RR^T> - y.q + (s/2)|q|^2          p1 = 2<C,RD^T> - y.q1 + s q.q1
 *   p2 = <C,DD^T> - y.q2 + (s/2)|q1|^2 + s q.q2     p3 = s q1.q2     p4 = (s/2)|q2|^2      */
void oracle_linesearch(const oracle_problem *P, const double *y, double sigma, const double *R,
                       const double *D, int32_t r, double *p) {
  size_t mm = (size_t)(P->m > 0 ? P->m : 1);
  double *q = (double *)malloc(sizeof(double) * mm), *q1 = (double *)malloc(sizeof(double) * mm),
         *q2 = (double *)malloc(sizeof(double) * mm);
  oracle_A_op(P, R, r, q);
  oracle_A_sym(P, R, D, r, q1); /* <A_i, RD^T+DR^T>/2 */
  oracle_A_op(P, D, r, q2);
  double yq = 0, yq1 = 0, yq2 = 0, qq = 0, qq1 = 0, qq2 = 0, q1q1 = 0, q1q2 = 0, q2q2 = 0;
  for (int64_t i = 0; i < P->m; ++i) {
    q[i] -= P->b[i];
    q1[i] *= 2.0;
    yq += y[i] * q[i]; yq1 += y[i] * q1[i]; yq2 += y[i] * q2[i];
    qq += q[i] * q[i]; qq1 += q[i] * q1[i]; qq2 += q[i] * q2[i];
    q1q1 += q1[i] * q1[i]; q1q2 += q1[i] * q2[i]; q2q2 += q2[i] * q2[i];
  }
  double cRR = oracle_inner_C(P, R, R, r), cRD = oracle_inner_C(P, R, D, r), cDD = oracle_inner_C(P, D, D, r);
  p[0] = cRR - yq + 0.5 * sigma * qq;
  p[1] = 2.0 * cRD - yq1 + sigma * qq1;
  p[2] = cDD - yq2 + 0.5 * sigma * q1q1 + sigma * qq2;
  p[3] = sigma * q1q2;
  p[4] = 0.5 * sigma * q2q2;
  free(q); free(q1); free(q2);
}

/* ||C_total||_F  (denominator of eq. 77 term 2).  Sparse part assumes coalesced
 * entries; the low-rank part is expanded exactly:
 * ||C + U S U^T||_F^2 = ||C||^2 + 2 sum_p s_p u_p^T C u_p + sum_pq s_p s_q (u_p^T u_q)^2. */
double oracle_normC_sq(const oracle_problem *P) {
  double s = 0.0;
  for (int64_t e = 0; e < P->nnzC; ++e) {
    double c = P->C_val[e];
    s += (P->C_row[e] == P->C_col[e] ? 1.0 : 2.0) * c * c;
  }
  for (int32_t p = 0; p < P->pC; ++p) {
    const double *u = P->C_U + (int64_t)p * P->n;
    double uCu = 0.0;
    for (int64_t e = 0; e < P->nnzC; ++e) {
      int64_t j = P->C_row[e], k = P->C_col[e];
      uCu += (j == k ? 1.0 : 2.0) * P->C_val[e] * u[j] * u[k];
    }
    s += 2.0 * P->C_s[p] * uCu;
    for (int32_t q = 0; q < P->pC; ++q) {
      const double *v = P->C_U + (int64_t)q * P->n;
      double uv = 0.0;
      for (int64_t j = 0; j < P->n; ++j) uv += u[j] * v[j];
      s += P->C_s[p] * P->C_s[q] * uv * uv;
    }
  }
  return s;
}
