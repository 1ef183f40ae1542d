/* alora_c_driver.c -- a plain C (C99) caller of the C ABI in include/alora.h, compiled and run by
 * tests/test_gpu_c_abi.py:  create -> set_dual -> eval -> linesearch (cold, warm) -> smatvec (mu, NULL) ->
 * lanczos (1 and 3 pairs) -> solve -> destroy on a problem read from a binary file, printing the scalars the
 * Python test compares with the oracle.  Device memory comes from the CUDA runtime's C API; nothing else is used.
 *
 * file layout (little endian): int64 n, m, nnzC, nnzA, r; then C_row[int32 nnzC], C_col, C_val[double],
 * A_ptr[int64 m+1], A_row[int32 nnzA], A_col, A_val[double], b[double m], y[double m], sigma[double 1],
 * R[double n*r], D[double n*r], V[double n]. */
#include <cuda_runtime_api.h>
#include <stdint.h>
#include <stdio.h>
#include <stdlib.h>

#include "alora.h"

#define CHECK(call)                                                                          \
  do {                                                                                       \
    alora_status st_ = (call);                                                               \
    if (st_ != ALORA_OK && st_ != ALORA_ENOTCONV) {                                           \
      fprintf(stderr, "%s -> %s: %s\n", #call, alora_strerror(st_), alora_last_error(ctx));  \
      return 2;                                                                              \
    }                                                                                        \
  } while (0)

static void *rd(FILE *f, size_t bytes) {
  void *p = malloc(bytes ? bytes : 1);
  if (bytes && fread(p, 1, bytes, f) != bytes) { fprintf(stderr, "short read\n"); exit(3); }
  return p;
}
static void *dev(const void *h, size_t bytes) {
  void *d = NULL;
  if (cudaMalloc(&d, bytes ? bytes : 16) != cudaSuccess) { fprintf(stderr, "cudaMalloc failed\n"); exit(4); }
  if (h && bytes) cudaMemcpy(d, h, bytes, cudaMemcpyHostToDevice);
  return d;
}

int main(int argc, char **argv) {
  alora_ctx *ctx = NULL;
  int64_t hdr[5];
  FILE *f;
  if (argc < 2 || !(f = fopen(argv[1], "rb"))) { fprintf(stderr, "usage: %s problem.bin\n", argv[0]); return 1; }
  if (fread(hdr, 8, 5, f) != 5) return 3;
  const int64_t n = hdr[0], m = hdr[1], nnzC = hdr[2], nnzA = hdr[3];
  const int32_t r = (int32_t)hdr[4];
  alora_problem P;
  P.n = n; P.m = m; P.nnzC = nnzC; P.nnzA = nnzA; P.pC = 0; P.C_U = NULL; P.C_s = NULL;
  P.C_row = rd(f, 4 * nnzC); P.C_col = rd(f, 4 * nnzC); P.C_val = rd(f, 8 * nnzC);
  P.A_ptr = rd(f, 8 * (m + 1)); P.A_row = rd(f, 4 * nnzA); P.A_col = rd(f, 4 * nnzA); P.A_val = rd(f, 8 * nnzA);
  P.b = rd(f, 8 * m);
  double *y = rd(f, 8 * m), *sigma = rd(f, 8), *R = rd(f, 8 * n * r), *D = rd(f, 8 * n * r), *V = rd(f, 8 * n);
  fclose(f);

  CHECK(alora_create(&P, ALORA_F64, 0, NULL, &ctx));
  double *y_d = dev(y, 8 * m), *R_d = dev(R, 8 * n * r), *D_d = dev(D, 8 * n * r), *V_d = dev(V, 8 * n);
  double *G_d = dev(NULL, 8 * n * r), *z_d = dev(NULL, 8 * m), *W_d = dev(NULL, 8 * n), *lam_d = dev(NULL, 8 * m);
  double *U_d = dev(NULL, 8 * n * 3);
  double st[8], p[5], pw[5], vw = 0.0, vw0 = 0.0, theta[3], resid[3];
  int32_t pf = 0, ku = 0;
  int64_t info[16];

  CHECK(alora_set_dual(ctx, y_d, *sigma));
  CHECK(alora_eval(ctx, R_d, r, r, G_d, z_d, st));
  printf("f %.17g\ncx %.17g\nyq %.17g\nqq %.17g\ngg %.17g\ngr %.17g\n", st[0], st[1], st[2], st[3], st[4], st[5]);
  CHECK(alora_linesearch(ctx, R_d, D_d, r, r, 0, p));
  CHECK(alora_linesearch(ctx, R_d, D_d, r, r, 1, pw));
  printf("p %.17g %.17g %.17g %.17g %.17g\n", p[0], p[1], p[2], p[3], p[4]);
  printf("pw %.17g %.17g %.17g %.17g %.17g\n", pw[0], pw[1], pw[2], pw[3], pw[4]);
  CHECK(alora_get_lambda(ctx, lam_d));
  CHECK(alora_smatvec(ctx, lam_d, V_d, 1, W_d, &vw));
  CHECK(alora_smatvec(ctx, NULL, V_d, 1, W_d, &vw0));
  printf("vw %.17g\nvw0 %.17g\n", vw, vw0);
  CHECK(alora_lanczos(ctx, lam_d, 300, 1e-8, 42, 1, theta, NULL, &pf, &ku, resid));
  printf("theta1 %.17g k %d found %d\n", theta[0], (int)ku, (int)pf);
  CHECK(alora_lanczos(ctx, NULL, 300, 1e-8, 42, 3, theta, U_d, &pf, &ku, resid));
  printf("theta3 %.17g %.17g %.17g found %d\n", theta[0], theta[1], theta[2], (int)pf);
  /* error path: warm line search without an evaluation of that pointer */
  printf("warm_without_eval %d\n", (int)alora_linesearch(ctx, D_d, R_d, r, r, 1, pw));
  /* Algorithm 1 from (R, y = 0) */
  {
    alora_params prm;
    alora_result res;
    int32_t rr = r;
    double sg = *sigma;
    double *Rs_d = dev(NULL, 8 * n * 64);
    alora_default_params(&prm);
    prm.eps = 1e-6;
    cudaMemcpy(Rs_d, R, 8 * n * r, cudaMemcpyHostToDevice);
    cudaMemset(y_d, 0, 8 * m);
    CHECK(alora_solve(ctx, &prm, Rs_d, &rr, 64, y_d, &sg, NULL, 0, &res));
    printf("solve converged %d outer %d r %d kkt %.3e %.3e %.3e\n", res.converged, res.outer_iters, (int)rr, res.kkt[0],
           res.kkt[1], res.kkt[2]);
    CHECK(alora_set_dual(ctx, y_d, sg));
    CHECK(alora_eval(ctx, Rs_d, rr, rr, NULL, NULL, st));
    printf("solve_cx %.17g\n", st[1]);
    cudaFree(Rs_d);
  }
  CHECK(alora_info(ctx, info));
  printf("class %d launches %lld\n", (int)info[0], (long long)info[7]);
  alora_destroy(ctx);
  cudaFree(y_d); cudaFree(R_d); cudaFree(D_d); cudaFree(V_d); cudaFree(G_d); cudaFree(z_d); cudaFree(W_d); cudaFree(lam_d); cudaFree(U_d);
  return 0;
}
