// alora_solve.cu -- the host-side driver pieces that exercise the hot-path kernels end to end
// (SURVEY.md 8a rows a7, a8): Lanczos with full re-orthogonalisation for lambda_min(S(mu)), and the
// ALORA loop of Algorithm 1 with the readings of DESIGN.md: L-BFGS(5) directions,
// exact quartic line search, rank growth along the most negative eigenvector with the closed-form
// step, rank shrink through the spectrum of R^T R, dual update, sigma schedule and the KKT stop of
// eq. 77.  All vector work runs in CUDA kernels on the ctx stream; the host keeps
// only scalars, the Lanczos tridiagonal and r x r matrices.  Written independently of the test oracle
// (same algorithm, no shared code).
#include <algorithm>
#include <chrono>
#include <cmath>
#include <cstring>

#include "alora_internal.h"

namespace alora {

// ---------------------------------------------------------------------------------------------
// BLAS-1 style kernels on flat arrays (fp64 accumulation, ordered two-stage reductions)
// ---------------------------------------------------------------------------------------------
constexpr int kRedBlocks = 592;  // 148 SMs x 4

template <typename TX, typename TY>
__global__ void __launch_bounds__(kBlock) k_dots3(int64_t N, const TX* x0, const TY* y0, const TX* x1, const TY* y1,
                                                  const TX* x2, const TY* y2, int nd, double* part) {
  double st[3] = {0.0, 0.0, 0.0};
  for (int64_t i = (int64_t)blockIdx.x * kBlock + threadIdx.x; i < N; i += (int64_t)gridDim.x * kBlock) {
    st[0] += (double)x0[i] * (double)y0[i];
    if (nd > 1) st[1] += (double)x1[i] * (double)y1[i];
    if (nd > 2) st[2] += (double)x2[i] * (double)y2[i];
  }
  block_reduce_store<3>(st, part + (int64_t)blockIdx.x * kNStat);
}

__global__ void k_reduce_rows(const double* part, int nrows, double* out) {  // ordered second stage
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  for (int s = warp; s < kNStat; s += kBlock / 32) {
    double v = 0.0;
    for (int i = lane; i < nrows; i += 32) v += part[(int64_t)i * kNStat + s];
    v = warp_sum(v);
    if (lane == 0) out[s] = v;
  }
}

// Element-wise passes: 16-byte packs over the aligned bulk (when both arrays are 16-byte aligned), scalars for the tail.
template <typename T, bool READ_Y, typename F> __device__ __forceinline__ void ew2(int64_t N, const T* x, T* y, F f) {   // y[i] = f(x[i], y[i])
  constexpr int VEC = 16 / (int)sizeof(T);
  const bool al = (((uintptr_t)x | (uintptr_t)y) & 15) == 0;
  const int64_t nv = al ? N / VEC : 0;
  const int64_t tid = (int64_t)blockIdx.x * blockDim.x + threadIdx.x, nth = (int64_t)gridDim.x * blockDim.x;
  for (int64_t i = tid; i < nv; i += 2 * nth) {   // two packs per thread in flight (the grid is four blocks per SM, see ew_grid)
    const int64_t i1 = i + nth;
    const bool two = i1 < nv;
    const Pack<T, VEC> xv0 = reinterpret_cast<const Pack<T, VEC>*>(x)[i];
    Pack<T, VEC> xv1 = xv0, yv0, yv1;
    if (two) xv1 = reinterpret_cast<const Pack<T, VEC>*>(x)[i1];
    if (READ_Y) { yv0 = reinterpret_cast<Pack<T, VEC>*>(y)[i]; if (two) yv1 = reinterpret_cast<Pack<T, VEC>*>(y)[i1]; }
#pragma unroll
    for (int k = 0; k < VEC; ++k) { yv0.v[k] = f(xv0.v[k], READ_Y ? yv0.v[k] : T(0)); yv1.v[k] = f(xv1.v[k], READ_Y ? yv1.v[k] : T(0)); }
    reinterpret_cast<Pack<T, VEC>*>(y)[i] = yv0;
    if (two) reinterpret_cast<Pack<T, VEC>*>(y)[i1] = yv1;
  }
  for (int64_t i = nv * VEC + tid; i < N; i += nth) y[i] = f(x[i], READ_Y ? y[i] : T(0));
}
template <typename T> __global__ void k_axpy(int64_t N, double a, const T* x, T* y) {  // y += a x
  ew2<T, true>(N, x, y, [a](T xv, T yv) { return (T)((double)yv + a * (double)xv); });
}
template <typename T> __global__ void k_scale_copy(int64_t N, double a, const T* x, T* y) {  // y = a x
  ew2<T, false>(N, x, y, [a](T xv, T) { return (T)(a * (double)xv); });
}
template <typename T> __global__ void k_scale(int64_t N, double a, T* y) {  // y *= a
  ew2<T, false>(N, y, y, [a](T xv, T) { return (T)(a * (double)xv); });
}
// L-BFGS pair: S = alpha D, Y = G - Gprev, and the sums S.Y, S.S, Y.Y in the same pass
template <typename T>
__global__ void __launch_bounds__(kBlock) k_make_pair(int64_t N, double alpha, const T* D, const T* G, const T* Gp,
                                                      T* S, T* Y, double* part) {
  double st[3] = {0.0, 0.0, 0.0};
  for (int64_t i = (int64_t)blockIdx.x * kBlock + threadIdx.x; i < N; i += (int64_t)gridDim.x * kBlock) {
    const T s = (T)(alpha * (double)D[i]);
    const T yv = (T)((double)G[i] - (double)Gp[i]);
    S[i] = s; Y[i] = yv;
    st[0] += (double)s * (double)yv; st[1] += (double)s * (double)s; st[2] += (double)yv * (double)yv;
  }
  block_reduce_store<3>(st, part + (int64_t)blockIdx.x * kNStat);
}
// ---- fused L-BFGS passes ("L-BFGS in two passes") ----------------------------------------
// The two-loop recursion only ever forms linear combinations of g, S_j, Y_j, so the direction is
//   d = cg g + sum_j cs_j S_j + sum_j cy_j Y_j
// with coefficients that follow from the dot products S_j.g, Y_j.g and the Gram blocks S_i.Y_j, Y_i.Y_j.  The Gram
// blocks change by one row / column per iteration (the new pair).  So an iteration needs two passes over the
// vectors instead of 4m + 6: k_lbfgs_dots (build the new pair, all new dot products) and k_lbfgs_combine.
constexpr int kLbMax = 8;            // pairs the fused path handles (memory <= kLbMax - 1)
constexpr int kMemMax = 16;          // largest lbfgs_mem (larger values are clamped); sizes SolveWorkspace::buf
constexpr int kLbW = 48;             // doubles per partial row (5 * kLbMax + 1 sums, padded)
struct LbVecs { const void* S[kLbMax]; const void* Y[kLbMax]; };
struct LbCoef { double cg; double cs[kLbMax]; double cy[kLbMax]; };

// Builds S_new = alpha D, Y_new = G - Gp into the LAST listed pair (if have_new) and sums, for the np listed pairs j:
//   [j] S_j.G   [np + j] Y_j.G   [2np + j] S_new.Y_j   [3np + j] S_j.Y_new   [4np + j] Y_new.Y_j   [5np] S_new.S_new
// (the last four only if have_new).  Partial rows of kLbW doubles per block; the block that finishes last adds
// them in block order into out[kLbW].
// The two halves of a block (threads 0..127 / 128..255) take the same 128 packs of an iteration and the even / odd pairs
// of the list, so a thread carries the sums of at most (NP + 1) / 2 pairs: about 70 registers and three blocks per SM
// instead of 128 - 142 registers and one or two (ncu, config 4 inside alora_solve: 3.2 TB/s with every product in fp64,
// 4.3 TB/s with pack-local sums, both bound by registers / the fp64 pipe rather than HBM; over 40 % of the solve's GPU
// time).  G, D, Gp are read by both halves (the second read hits L1 / L2).
// The VEC products of a pack are summed in the vector type (fp32 contexts: FFMA) and enter the fp64 sums once per pack:
// the library's precision model -- products and short local sums in the context type, everything that crosses rows in
// fp64.
template <typename T, int NP, int PAR>
__device__ __forceinline__ void lbfgs_dots_half(int64_t nv, int have_new, double alpha, const T* D, const T* G, const T* Gp, const LbVecs& v,
                                                T* Snew, T* Ynew, double (*sm)[kBlock / 32]) {
  constexpr int VEC = 16 / (int)sizeof(T), HB = kBlock / 2;
  constexpr int NH = (NP - PAR + 1) / 2;        // pairs j = PAR, PAR + 2, ... < NP
  double sg[NH > 0 ? NH : 1], yg[NH > 0 ? NH : 1], sny[NH > 0 ? NH : 1], syn[NH > 0 ? NH : 1], yyn[NH > 0 ? NH : 1], ss = 0.0;
#pragma unroll
  for (int h = 0; h < NH; ++h) { sg[h] = yg[h] = sny[h] = syn[h] = yyn[h] = 0.0; }
  const int tx = threadIdx.x % HB;
  for (int64_t i = (int64_t)blockIdx.x * HB + tx; i < nv; i += (int64_t)gridDim.x * HB) {
    const Pack<T, VEC> g = reinterpret_cast<const Pack<T, VEC>*>(G)[i];
    Pack<T, VEC> sn, yn;
    if (have_new) {
      const Pack<T, VEC> d = reinterpret_cast<const Pack<T, VEC>*>(D)[i], gp = reinterpret_cast<const Pack<T, VEC>*>(Gp)[i];
#pragma unroll
      for (int k = 0; k < VEC; ++k) { sn.v[k] = (T)(alpha * (double)d.v[k]); yn.v[k] = (T)((double)g.v[k] - (double)gp.v[k]); }
      if (PAR == 0) {
        reinterpret_cast<Pack<T, VEC>*>(Snew)[i] = sn;
        reinterpret_cast<Pack<T, VEC>*>(Ynew)[i] = yn;
      }
    }
#pragma unroll
    for (int h = 0; h < NH; ++h) {
      const int j = PAR + 2 * h;
      Pack<T, VEC> sj, yj;
      if (have_new && j == NP - 1) { sj = sn; yj = yn; }
      else { sj = reinterpret_cast<const Pack<T, VEC>*>(v.S[j])[i]; yj = reinterpret_cast<const Pack<T, VEC>*>(v.Y[j])[i]; }
      T a0 = T(0), a1 = T(0), a2 = T(0), a3 = T(0), a4 = T(0);
#pragma unroll
      for (int k = 0; k < VEC; ++k) {
        a0 = fma(sj.v[k], g.v[k], a0); a1 = fma(yj.v[k], g.v[k], a1);
        if (have_new) { a2 = fma(sn.v[k], yj.v[k], a2); a3 = fma(sj.v[k], yn.v[k], a3); a4 = fma(yn.v[k], yj.v[k], a4); }
      }
      sg[h] += (double)a0; yg[h] += (double)a1;
      if (have_new) { sny[h] += (double)a2; syn[h] += (double)a3; yyn[h] += (double)a4; }
    }
    if (PAR == 0 && have_new) {
      T a = T(0);
#pragma unroll
      for (int k = 0; k < VEC; ++k) a = fma(sn.v[k], sn.v[k], a);
      ss += (double)a;
    }
  }
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  auto put = [&](int slot, double val) { const double t = warp_sum(val); if (lane == 0) sm[slot][warp] = t; };
#pragma unroll
  for (int h = 0; h < NH; ++h) {
    const int j = PAR + 2 * h;
    put(j, sg[h]); put(NP + j, yg[h]); put(2 * NP + j, sny[h]); put(3 * NP + j, syn[h]); put(4 * NP + j, yyn[h]);
  }
  if (PAR == 0) put(5 * NP, ss);
}

template <typename T, int NP>
__global__ void __launch_bounds__(kBlock, 3) k_lbfgs_dots(int64_t N, int have_new, double alpha, const T* D, const T* G, const T* Gp,
                                                          LbVecs v, T* Snew, T* Ynew, double* part, double* out,
                                                          unsigned int* ticket) {
  constexpr int VEC = 16 / (int)sizeof(T);
  __shared__ double sm[kLbW][kBlock / 32];
  __shared__ unsigned int s_last;
  for (int t = threadIdx.x; t < kLbW * (kBlock / 32); t += kBlock) (&sm[0][0])[t] = 0.0;   // a warp fills only its half's slots
  __syncthreads();
  const int64_t nv = N / VEC;
  if (threadIdx.x < kBlock / 2) lbfgs_dots_half<T, NP, 0>(nv, have_new, alpha, D, G, Gp, v, Snew, Ynew, sm);
  else lbfgs_dots_half<T, NP, 1>(nv, have_new, alpha, D, G, Gp, v, Snew, Ynew, sm);
  __syncthreads();
  if (threadIdx.x < kLbW) {
    double t = 0.0;
    if (threadIdx.x <= 5 * NP)
      for (int wv = 0; wv < kBlock / 32; ++wv) t += sm[threadIdx.x][wv];
    part[(int64_t)blockIdx.x * kLbW + threadIdx.x] = t;
  }
  __threadfence();
  __syncthreads();
  if (threadIdx.x == 0) s_last = (atomicAdd(ticket, 1u) == gridDim.x - 1) ? 1u : 0u;
  __syncthreads();
  if (!s_last) return;
  __threadfence();
  // ordered final sum: thread t owns column t % kLbW and the rows t / kLbW, + 5, ... (kBlock / kLbW = 5 slices)
  __shared__ double fin[kBlock];
  constexpr int NSL = kBlock / kLbW;
  const int col = threadIdx.x % kLbW, sl = threadIdx.x / kLbW;
  double t = 0.0;
  if (sl < NSL) {
    int b = sl;
    for (; b + 3 * NSL < (int)gridDim.x; b += 4 * NSL) {
      const double v0 = __ldcg(part + (int64_t)b * kLbW + col), v1 = __ldcg(part + (int64_t)(b + NSL) * kLbW + col);
      const double v2 = __ldcg(part + (int64_t)(b + 2 * NSL) * kLbW + col), v3 = __ldcg(part + (int64_t)(b + 3 * NSL) * kLbW + col);
      t += v0; t += v1; t += v2; t += v3;
    }
    for (; b < (int)gridDim.x; b += NSL) t += __ldcg(part + (int64_t)b * kLbW + col);
  }
  fin[threadIdx.x] = t;
  __syncthreads();
  if (threadIdx.x < kLbW) {
    double u = 0.0;
    for (int k = 0; k < NSL; ++k) u += fin[k * kLbW + threadIdx.x];
    out[threadIdx.x] = u;
  }
  if (threadIdx.x == 0) *ticket = 0u;
}

// D = cg G + sum_j cs_j S_j + cy_j Y_j   (one pass, fp64 accumulation, rounded once)
template <typename T, int NP>
__global__ void __launch_bounds__(kBlock) k_lbfgs_combine(int64_t N, const T* G, LbVecs v, LbCoef c, T* D) {
  constexpr int VEC = 16 / (int)sizeof(T);
  const int64_t nv = N / VEC;
  for (int64_t i = (int64_t)blockIdx.x * kBlock + threadIdx.x; i < nv; i += (int64_t)gridDim.x * kBlock) {
    const Pack<T, VEC> g = reinterpret_cast<const Pack<T, VEC>*>(G)[i];
    double acc[VEC];
#pragma unroll
    for (int k = 0; k < VEC; ++k) acc[k] = c.cg * (double)g.v[k];
#pragma unroll
    for (int j = 0; j < NP; ++j) {
      const Pack<T, VEC> sj = reinterpret_cast<const Pack<T, VEC>*>(v.S[j])[i], yj = reinterpret_cast<const Pack<T, VEC>*>(v.Y[j])[i];
#pragma unroll
      for (int k = 0; k < VEC; ++k) acc[k] += c.cs[j] * (double)sj.v[k] + c.cy[j] * (double)yj.v[k];
    }
    Pack<T, VEC> o;
#pragma unroll
    for (int k = 0; k < VEC; ++k) o.v[k] = (T)acc[k];
    reinterpret_cast<Pack<T, VEC>*>(D)[i] = o;
  }
}
// w -= a v + b u   (Lanczos three-term recurrence); a = *a_dev is <v, S v> left on the device by the matvec
template <typename T> __global__ void k_axpy2(int64_t N, const double* a_dev, const T* v, double b, const T* u, T* w) {
  const double a = *a_dev;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += (int64_t)gridDim.x * blockDim.x)
    w[i] = (T)((double)w[i] - a * (double)v[i] - (u ? b * (double)u[i] : 0.0));
}
// c[j] = <V_j, w> for j < k: V is k x N (row j contiguous).  blockIdx.y takes kBasisJB consecutive vectors j (w is read
// once for all of them, 16-byte loads when N is a multiple of the pack), nchunk blocks per group leave partial sums;
// the block that draws the last ticket adds the chunks of every j in order (no separate reduction launch).
// (Before: one vector per blockIdx.y and 4-byte loads -- w was re-read for every j and the kernel ran at 2.8 TB/s.)
constexpr int kBasisJB = 4;
template <typename T>
__global__ void __launch_bounds__(kBlock) k_basis_dots(int64_t N, const T* V, const T* w, double* part, int nchunk, int k,
                                                       double* c, unsigned int* ticket) {
  constexpr int VEC = 16 / (int)sizeof(T), JB = kBasisJB;
  const int j0 = blockIdx.y * JB, nj = min(JB, k - j0);
  double st[JB];
#pragma unroll
  for (int q = 0; q < JB; ++q) st[q] = 0.0;
  if (N % VEC == 0) {
    const int64_t nv = N / VEC;
    for (int64_t i = (int64_t)blockIdx.x * kBlock + threadIdx.x; i < nv; i += (int64_t)gridDim.x * kBlock) {
      const Pack<T, VEC> wv = reinterpret_cast<const Pack<T, VEC>*>(w)[i];
      Pack<T, VEC> vv[JB];
#pragma unroll
      for (int q = 0; q < JB; ++q) if (q < nj) vv[q] = reinterpret_cast<const Pack<T, VEC>*>(V + (int64_t)(j0 + q) * N)[i];
#pragma unroll
      for (int q = 0; q < JB; ++q) if (q < nj) {
        T a = T(0);
#pragma unroll
        for (int e = 0; e < VEC; ++e) a = fma(vv[q].v[e], wv.v[e], a);
        st[q] += (double)a;
      }
    }
  } else {
    for (int64_t i = (int64_t)blockIdx.x * kBlock + threadIdx.x; i < N; i += (int64_t)gridDim.x * kBlock) {
      const double wi = (double)w[i];
#pragma unroll
      for (int q = 0; q < JB; ++q) if (q < nj) st[q] += (double)V[(int64_t)(j0 + q) * N + i] * wi;
    }
  }
  __shared__ double sm[JB][kBlock / 32];
  __shared__ unsigned int s_last;
#pragma unroll
  for (int q = 0; q < JB; ++q) { const double v = warp_sum(st[q]); if ((threadIdx.x & 31) == 0) sm[q][threadIdx.x >> 5] = v; }
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int q = 0; q < nj; ++q) {
      double t = 0.0;
      for (int wv = 0; wv < kBlock / 32; ++wv) t += sm[q][wv];
      part[(int64_t)(j0 + q) * nchunk + blockIdx.x] = t;
    }
    __threadfence();
    s_last = (atomicAdd(ticket, 1u) == gridDim.x * gridDim.y - 1) ? 1u : 0u;
  }
  __syncthreads();
  if (!s_last) return;
  __threadfence();
  for (int jj = threadIdx.x >> 5; jj < k; jj += kBlock / 32) {   // a warp per vector: lanes over the chunks, then an ordered warp sum
    double t = 0.0;
    for (int i = threadIdx.x & 31; i < nchunk; i += 32) t += __ldcg(part + (int64_t)jj * nchunk + i);
    t = warp_sum(t);
    if ((threadIdx.x & 31) == 0) c[jj] = t;
  }
  if (threadIdx.x == 0) *ticket = 0u;
}
// out[i] = beta*out[i] + sign * sum_j c[j] V[j][i]    (c on the device); nrm != nullptr: also ||out||^2 (ordered
// two-stage sum, the block that finishes last adds the per-block partials)
template <typename T>
__global__ void __launch_bounds__(kBlock) k_basis_combine(int64_t N, int k, const T* V, const double* c, double beta, double sign, T* out,
                                                          double* part, double* nrm, unsigned int* ticket) {
  double st[1] = {0.0};
  constexpr int VEC = 16 / (int)sizeof(T);
  if (N % VEC == 0) {   // 16-byte loads, four basis vectors in flight per thread (the scalar form ran at 3.1 TB/s)
    const int64_t nv = N / VEC;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < nv; i += (int64_t)gridDim.x * blockDim.x) {
      double t[VEC];
#pragma unroll
      for (int e = 0; e < VEC; ++e) t[e] = 0.0;
      int j = 0;
      for (; j + 4 <= k; j += 4) {
        Pack<T, VEC> vv[4];
#pragma unroll
        for (int q = 0; q < 4; ++q) vv[q] = reinterpret_cast<const Pack<T, VEC>*>(V + (int64_t)(j + q) * N)[i];
#pragma unroll
        for (int q = 0; q < 4; ++q) {
          const double cj = __ldg(c + j + q);
#pragma unroll
          for (int e = 0; e < VEC; ++e) t[e] += cj * (double)vv[q].v[e];
        }
      }
      for (; j < k; ++j) {
        const Pack<T, VEC> vv = reinterpret_cast<const Pack<T, VEC>*>(V + (int64_t)j * N)[i];
        const double cj = __ldg(c + j);
#pragma unroll
        for (int e = 0; e < VEC; ++e) t[e] += cj * (double)vv.v[e];
      }
      Pack<T, VEC> o;
      if (beta != 0.0) o = reinterpret_cast<const Pack<T, VEC>*>(out)[i];
#pragma unroll
      for (int e = 0; e < VEC; ++e) {
        o.v[e] = (T)((beta != 0.0 ? beta * (double)o.v[e] : 0.0) + sign * t[e]);
        st[0] += (double)o.v[e] * (double)o.v[e];
      }
      reinterpret_cast<Pack<T, VEC>*>(out)[i] = o;
    }
  } else {
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += (int64_t)gridDim.x * blockDim.x) {
      double t = 0.0;
      for (int j = 0; j < k; ++j) t += c[j] * (double)V[(int64_t)j * N + i];
      const T o = (T)((beta != 0.0 ? beta * (double)out[i] : 0.0) + sign * t);
      out[i] = o;
      st[0] += (double)o * (double)o;
    }
  }
  if (!nrm) return;
  __shared__ double sm[kBlock / 32];
  __shared__ unsigned int s_last;
  const double v = warp_sum(st[0]);
  if ((threadIdx.x & 31) == 0) sm[threadIdx.x >> 5] = v;
  __syncthreads();
  if (threadIdx.x == 0) {
    double t = 0.0;
    for (int wv = 0; wv < kBlock / 32; ++wv) t += sm[wv];
    part[blockIdx.x] = t;
    __threadfence();
    s_last = (atomicAdd(ticket, 1u) == gridDim.x - 1) ? 1u : 0u;
  }
  __syncthreads();
  if (!s_last) return;
  __threadfence();
  if (threadIdx.x < 32) {
    double t = 0.0;
    for (int i = threadIdx.x; i < (int)gridDim.x; i += 32) t += __ldcg(part + i);   // lane-strided, then an ordered warp sum
    t = warp_sum(t);
    if (threadIdx.x == 0) { *nrm = t; *ticket = 0u; }
  }
}
// v0[i] = counter_uniform(seed, i) in (-1,1): splitmix64-style hash, integer arithmetic only
template <typename T> __global__ void k_counter_uniform(int64_t N, uint64_t seed, T* v) {
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += (int64_t)gridDim.x * blockDim.x) {
    uint64_t x = (uint64_t)i + seed * 0x9E3779B97F4A7C15ull;
    x = (x ^ (x >> 30)) * 0xBF58476D1CE4E5B9ull;
    x = (x ^ (x >> 27)) * 0x94D049BB133111EBull;
    x = x ^ (x >> 31);
    v[i] = (T)(((double)(x >> 11) + 0.5) * (2.0 / 9007199254740992.0) - 1.0);
  }
}
// repack rows: dst (ld_d) <- src (ld_s), columns [0, r) copied, [r, ld_d) zeroed
template <typename T> __global__ void k_repack(int64_t n, int r, const T* src, int64_t ld_s, T* dst, int64_t ld_d) {
  const int64_t N = n * ld_d;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += (int64_t)gridDim.x * blockDim.x) {
    const int64_t row = i / ld_d; const int c = (int)(i - row * ld_d);
    dst[i] = c < r ? src[row * ld_s + c] : T(0);
  }
}
template <typename T> __global__ void k_set_col(int64_t n, int64_t ld, int col, double scale, const T* v, T* R) {
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x)
    R[i * ld + col] = (T)(scale * (double)v[i]);
}
// Gram matrix partials: part[block][i*r+j] = sum over the block's rows of R[row][i] R[row][j]
template <typename T> __global__ void k_gram(int64_t n, int r, const T* R, int64_t ld, double* part, int64_t rows_per_block) {
  const int64_t r0 = (int64_t)blockIdx.x * rows_per_block, r1 = min(n, r0 + rows_per_block);
  for (int p = threadIdx.x; p < r * r; p += blockDim.x) {
    const int i = p / r, j = p % r;
    double t = 0.0;
    for (int64_t row = r0; row < r1; ++row) t += (double)R[row * ld + i] * (double)R[row * ld + j];
    part[(int64_t)blockIdx.x * r * r + p] = t;
  }
}
__global__ void k_gram_reduce(const double* part, int nblk, int rr, double* M) {
  for (int p = blockIdx.x * blockDim.x + threadIdx.x; p < rr; p += gridDim.x * blockDim.x) {
    double t = 0.0;
    for (int bk = 0; bk < nblk; ++bk) t += part[(int64_t)bk * rr + p];
    M[p] = t;
  }
}
// dst[row][c] = sum_i src[row][i] Q[i*rk + c]  for c < rk; zero for rk <= c < ld_d
template <typename T>
__global__ void k_rotate(int64_t n, int r, int rk, const T* src, int64_t ld_s, const double* Q, T* dst, int64_t ld_d) {
  const int64_t N = n * ld_d;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += (int64_t)gridDim.x * blockDim.x) {
    const int64_t row = i / ld_d; const int c = (int)(i - row * ld_d);
    double t = 0.0;
    if (c < rk) for (int k = 0; k < r; ++k) t += (double)src[row * ld_s + k] * Q[k * rk + c];
    dst[i] = (T)t;
  }
}
// y <- y - sigma (z - b)   (Alg. 1 line 10)
__global__ void k_dual_update(int64_t m, double sigma, const double* z, const double* b, double* y) {
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < m; i += (int64_t)gridDim.x * blockDim.x)
    y[i] -= sigma * (z[i] - b[i]);
}
__global__ void k_lambda2(int64_t m, const double* y, const double* z, const double* b, double sigma, double* lam) {
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < m; i += (int64_t)gridDim.x * blockDim.x)
    lam[i] = y[i] - sigma * (z[i] - b[i]);
}

// ---------------------------------------------------------------------------------------------
// workspace
// ---------------------------------------------------------------------------------------------
struct SolveWorkspace {
  // Lanczos
  void* V = nullptr; int V_cap = 0;  // basis, V_cap x n
  void* w = nullptr;                 // n
  double* bd_part = nullptr; double* cvec = nullptr; int bd_chunks = 0;
  double* red_part = nullptr; double* red_out = nullptr;
  double* lb_part = nullptr; double* lb_out = nullptr;   // k_lbfgs_dots partial rows / result
  int occ_dots[kLbMax + 1] = {}, occ_comb[kLbMax + 1] = {};   // resident blocks per SM of k_lbfgs_dots / k_lbfgs_combine by pair count
  // solve
  static constexpr int kNBuf = 5 + 2 * (kMemMax + 1);   // R, G, D, Gprev, Rtmp + (mem + 1) slots each of S and Y
  void* buf[kNBuf] = {}; int nbuf = 0; int64_t buf_elems = 0;
  double* lam = nullptr; double* z = nullptr; double* zv = nullptr; void* ritz = nullptr;
  double* gram_part = nullptr; double* gram = nullptr; double* Qdev = nullptr;
  void* ritzp = nullptr; void* vtmp = nullptr; double* cab = nullptr;   // p_max > 1: Ritz vectors (4 x n), v_a + v_b, c_ab (11 x m)
};

void free_solve_workspace(alora_ctx* c) {
  if (!c->ws) return;
  // device memory belongs to the ctx pool (freed by alora_destroy); only the struct is ours
  delete c->ws;
  c->ws = nullptr;
}

}  // namespace alora

// ---------------------------------------------------------------------------------------------
// host numerics: tridiagonal eigenpair, cubic roots, Jacobi
// ---------------------------------------------------------------------------------------------
namespace alora {
namespace {

// number of eigenvalues of the tridiagonal (a, b) that are < x  (Sturm count)
int sturm_count(const std::vector<double>& a, const std::vector<double>& b, int k, double x) {
  int cnt = 0;
  double d = 1.0;
  for (int i = 0; i < k; ++i) {
    const double off = i ? b[i - 1] : 0.0;
    d = (a[i] - x) - (i ? off * off / d : 0.0);
    if (d == 0.0) d = 1e-300;
    if (d < 0.0) ++cnt;
  }
  return cnt;
}

// smallest eigenvalue (bisection) and its unit eigenvector (inverse iteration) of the k x k
// symmetric tridiagonal with diagonal a[0..k) and off-diagonal b[0..k-1)
// (j+1)-th smallest eigenvalue and its unit eigenvector; `prev`: eigenvectors already found (kept orthogonal to)
void tridiag_jth(const std::vector<double>& a, const std::vector<double>& b, int k, int j, double& theta,
                 std::vector<double>& s, const std::vector<std::vector<double>>& prev) {
  s.assign(k, 0.0);
  if (k == 1) { theta = a[0]; s[0] = 1.0; return; }
  double lo = a[0], hi = a[0], scale = 0.0;
  for (int i = 0; i < k; ++i) {
    const double rad = (i ? std::fabs(b[i - 1]) : 0.0) + (i + 1 < k ? std::fabs(b[i]) : 0.0);
    lo = std::min(lo, a[i] - rad); hi = std::max(hi, a[i] + rad);
    scale = std::max(scale, std::fabs(a[i]) + rad);
  }
  double l = lo, h = hi;
  for (int it = 0; it < 200 && h - l > 4e-16 * std::max(std::fabs(l), std::fabs(h)) + 1e-300; ++it) {
    const double mid = 0.5 * (l + h);
    if (mid <= l || mid >= h) break;
    if (sturm_count(a, b, k, mid) >= j + 1) h = mid; else l = mid;
  }
  theta = 0.5 * (l + h);
  // inverse iteration: (T - shift I) x = rhs with partial pivoting (shift nudged off the eigenvalue)
  const double shift = theta - 1e-13 * std::max(scale, 1e-300) - 1e-300;
  std::vector<double> x(k), dl(k), d(k), du(k), du2(k);
  for (int i = 0; i < k; ++i) x[i] = 1.0 + 0.01 * (((i + 31 * j) * 7919) % 13);
  for (int rep = 0; rep < 4; ++rep) {
    for (int i = 0; i < k; ++i) { d[i] = a[i] - shift; du[i] = i + 1 < k ? b[i] : 0.0; dl[i] = i + 1 < k ? b[i] : 0.0; du2[i] = 0.0; }
    // LU with partial pivoting on the tridiagonal (dgtsv style), applied to x
    for (int i = 0; i + 1 < k; ++i) {
      if (std::fabs(d[i]) >= std::fabs(dl[i])) {
        if (d[i] == 0.0) d[i] = 1e-300;
        const double f = dl[i] / d[i];
        d[i + 1] -= f * du[i];
        x[i + 1] -= f * x[i];
        du2[i] = 0.0;
      } else {
        const double f = d[i] / dl[i];
        d[i] = dl[i];
        const double t = d[i + 1];
        d[i + 1] = du[i] - f * t;
        du2[i] = i + 2 < k ? du[i + 1] : 0.0;
        if (i + 2 < k) du[i + 1] = -f * du2[i];
        du[i] = t;
        const double tx = x[i]; x[i] = x[i + 1]; x[i + 1] = tx - f * x[i + 1];
      }
    }
    if (d[k - 1] == 0.0) d[k - 1] = 1e-300;
    x[k - 1] /= d[k - 1];
    if (k > 1) x[k - 2] = (x[k - 2] - du[k - 2] * x[k - 1]) / d[k - 2];
    for (int i = k - 3; i >= 0; --i) x[i] = (x[i] - du[i] * x[i + 1] - du2[i] * x[i + 2]) / d[i];
    for (const auto& pv : prev) {   // close eigenvalues: stay orthogonal to the vectors already found
      double d0 = 0.0;
      for (int i = 0; i < k; ++i) d0 += pv[i] * x[i];
      for (int i = 0; i < k; ++i) x[i] -= d0 * pv[i];
    }
    double nrm = 0.0;
    for (int i = 0; i < k; ++i) nrm += x[i] * x[i];
    nrm = std::sqrt(nrm);
    if (!(nrm > 0.0) || !std::isfinite(nrm)) { for (int i = 0; i < k; ++i) x[i] = (i == j % k); nrm = 1.0; }
    for (int i = 0; i < k; ++i) x[i] /= nrm;
  }
  s = x;
}
void tridiag_smallest(const std::vector<double>& a, const std::vector<double>& b, int k, double& theta,
                      std::vector<double>& s) {
  tridiag_jth(a, b, k, 0, theta, s, {});
}

// real roots of c3 x^3 + c2 x^2 + c1 x + c0 (c3 != 0); a complex pair whose imaginary part is below
// 1e-8 * scale counts as a (double) real root
int cubic_real_roots(double c3, double c2, double c1, double c0, double out[3]) {
  const double b = c2 / c3, c = c1 / c3, d = c0 / c3;
  const double Q = (b * b - 3.0 * c) / 9.0, R = (2.0 * b * b * b - 9.0 * b * c + 27.0 * d) / 54.0;
  const double Q3 = Q * Q * Q;
  if (R * R < Q3) {
    const double th = std::acos(std::max(-1.0, std::min(1.0, R / std::sqrt(Q3))));
    const double sq = -2.0 * std::sqrt(Q);
    const double PI = 3.14159265358979323846;
    out[0] = sq * std::cos(th / 3.0) - b / 3.0;
    out[1] = sq * std::cos((th + 2.0 * PI) / 3.0) - b / 3.0;
    out[2] = sq * std::cos((th - 2.0 * PI) / 3.0) - b / 3.0;
    return 3;
  }
  const double A = -(R >= 0.0 ? 1.0 : -1.0) * std::cbrt(std::fabs(R) + std::sqrt(std::max(0.0, R * R - Q3)));
  const double B = A != 0.0 ? Q / A : 0.0;
  out[0] = (A + B) - b / 3.0;
  const double re = -0.5 * (A + B) - b / 3.0, im = 0.8660254037844386 * std::fabs(A - B);
  const double scale = std::max(1.0, std::max(std::fabs(out[0]), std::hypot(re, im)));
  if (im <= 1e-8 * scale) { out[1] = re; out[2] = re; return 3; }
  return 1;
}

// exact line search (reading 20): argmin over alpha > 0 of sum_k p_k alpha^k
double quartic_argmin(const double p[5], int* flag) {
  *flag = 0;
  if (p[4] == 0.0 && p[3] == 0.0) {
    if (p[2] > 0.0 && -p[1] / (2.0 * p[2]) > 0.0) return -p[1] / (2.0 * p[2]);
    *flag = 1; return 1.0;
  }
  double roots[3]; int nr;
  if (p[4] != 0.0) nr = cubic_real_roots(4.0 * p[4], 3.0 * p[3], 2.0 * p[2], p[1], roots);
  else {  // quadratic 3 p3 x^2 + 2 p2 x + p1
    const double qa = 3.0 * p[3], qb = 2.0 * p[2], qc = p[1], disc = qb * qb - 4.0 * qa * qc;
    if (disc < 0.0) nr = 0;
    else { const double sq = std::sqrt(disc); roots[0] = (-qb - sq) / (2.0 * qa); roots[1] = (-qb + sq) / (2.0 * qa); nr = 2; }
  }
  double cand[3]; int nc = 0;
  for (int i = 0; i < nr; ++i) {
    double a = roots[i];
    for (int it = 0; it < 2; ++it) {
      const double d1 = p[1] + a * (2.0 * p[2] + a * (3.0 * p[3] + a * 4.0 * p[4]));
      const double d2 = 2.0 * p[2] + a * (6.0 * p[3] + a * 12.0 * p[4]);
      if (d2 != 0.0) a -= d1 / d2;
    }
    if (a > 0.0) cand[nc++] = a;
  }
  if (!nc) { *flag = 1; return 1.0; }
  std::sort(cand, cand + nc);
  auto phi = [&](double a) { return p[0] + a * (p[1] + a * (p[2] + a * (p[3] + a * p[4]))); };
  double best = cand[0];
  for (int i = 1; i < nc; ++i)
    if (phi(cand[i]) < phi(best) - 1e-14 * (std::fabs(phi(best)) + std::fabs(p[0]))) best = cand[i];
  return best;
}

// cyclic Jacobi for a symmetric r x r matrix (row-major M, destroyed): eigenvalues ascending in mu,
// eigenvectors in the columns of Q (row-major r x r)
void jacobi_eigh(std::vector<double>& M, int r, std::vector<double>& mu, std::vector<double>& Q) {
  Q.assign((size_t)r * r, 0.0);
  for (int i = 0; i < r; ++i) Q[i * r + i] = 1.0;
  for (int sweep = 0; sweep < 60; ++sweep) {
    double off = 0.0, diag = 0.0;
    for (int i = 0; i < r; ++i) for (int j = 0; j < r; ++j) (i == j ? diag : off) += M[i * r + j] * M[i * r + j];
    if (off <= 1e-30 * diag || off == 0.0) break;
    for (int p = 0; p < r; ++p)
      for (int q = p + 1; q < r; ++q) {
        const double apq = M[p * r + q];
        if (apq == 0.0) continue;
        const double tau = (M[q * r + q] - M[p * r + p]) / (2.0 * apq);
        const double t = (tau >= 0.0 ? 1.0 : -1.0) / (std::fabs(tau) + std::sqrt(1.0 + tau * tau));
        const double cs = 1.0 / std::sqrt(1.0 + t * t), sn = t * cs;
        for (int k = 0; k < r; ++k) {
          const double mkp = M[k * r + p], mkq = M[k * r + q];
          M[k * r + p] = cs * mkp - sn * mkq; M[k * r + q] = sn * mkp + cs * mkq;
        }
        for (int k = 0; k < r; ++k) {
          const double mpk = M[p * r + k], mqk = M[q * r + k];
          M[p * r + k] = cs * mpk - sn * mqk; M[q * r + k] = sn * mpk + cs * mqk;
        }
        for (int k = 0; k < r; ++k) {
          const double qkp = Q[k * r + p], qkq = Q[k * r + q];
          Q[k * r + p] = cs * qkp - sn * qkq; Q[k * r + q] = sn * qkp + cs * qkq;
        }
      }
  }
  std::vector<int> order(r);
  for (int i = 0; i < r; ++i) order[i] = i;
  std::sort(order.begin(), order.end(), [&](int x, int y) { return M[x * r + x] < M[y * r + y]; });
  mu.resize(r);
  std::vector<double> Qs((size_t)r * r);
  for (int c = 0; c < r; ++c) {
    mu[c] = M[order[c] * r + order[c]];
    for (int k = 0; k < r; ++k) Qs[k * r + c] = Q[k * r + order[c]];
  }
  Q.swap(Qs);
}

// grid of the element-wise / streaming kernels: four blocks of 256 threads per SM are resident at once for every kernel of
// this file with <= 64 registers; with eight (the former value) the 40 - 44 register kernels (k_axpy, k_basis_combine) had six
// or five resident and ran a partial second wave (ncu: R += alpha D at 5.9 TB/s)
inline int ew_grid(alora_ctx* c, int64_t N) {
  return (int)std::max<int64_t>(1, std::min<int64_t>((N + 255) / 256, (int64_t)c->num_sms * 4));
}

}  // namespace
}  // namespace alora

// ---------------------------------------------------------------------------------------------
// device helpers with host results
// ---------------------------------------------------------------------------------------------
namespace alora {
namespace {

// Alg. 1 line 7 for p <= 4 directions, reading 29: minimise over S psd (p x p)
//   g(S) = sum_a theta_a S_aa + (sigma/2) s^T Hw s,   s = (S_ab)_{a<=b} row-major, Hw = H .* (w w^T), w_ab = 1 or 2,
// H[(ab),(cd)] = <c_ab, c_cd>, by projected gradient with step 1/L from S0 = diag(-theta_a / (sigma H[(aa),(aa)])).
// S row-major p x p out; returns g(S).
double growth_sdp_host(int p, const double* theta, const std::vector<double>& H, double sigma, std::vector<double>& S, int iters = 500) {
  const int np = p * (p + 1) / 2;
  std::vector<int> pa(np), pb(np);
  std::vector<double> wgt(np);
  { int t = 0; for (int a = 0; a < p; ++a) for (int b = a; b < p; ++b) { pa[t] = a; pb[t] = b; wgt[t] = a == b ? 1.0 : 2.0; ++t; } }
  auto Hw = [&](int i, int j) { return H[(size_t)i * np + j] * wgt[i] * wgt[j]; };
  // Lipschitz constant: sigma * lambda_max(D Hw D), D = diag(1 or 1/sqrt 2)
  std::vector<double> B((size_t)np * np), mu, Q;
  for (int i = 0; i < np; ++i) for (int j = 0; j < np; ++j)
    B[(size_t)i * np + j] = Hw(i, j) * (pa[i] == pb[i] ? 1.0 : M_SQRT1_2) * (pa[j] == pb[j] ? 1.0 : M_SQRT1_2);
  jacobi_eigh(B, np, mu, Q);
  const double L = sigma * std::max(mu[np - 1], 1e-300);
  S.assign((size_t)p * p, 0.0);
  for (int a = 0; a < p; ++a) {
    int idx = 0; for (int t = 0; t < np; ++t) if (pa[t] == a && pb[t] == a) idx = t;
    const double haa = H[(size_t)idx * np + idx];
    S[a * p + a] = haa > 0.0 ? std::max(0.0, -theta[a] / (sigma * haa)) : 0.0;
  }
  std::vector<double> sv(np), tv(np), G((size_t)p * p);
  auto gval = [&]() {
    for (int t = 0; t < np; ++t) sv[t] = S[pa[t] * p + pb[t]];
    double q = 0.0;
    for (int i = 0; i < np; ++i) { double r2 = 0.0; for (int j = 0; j < np; ++j) r2 += Hw(i, j) * sv[j]; q += sv[i] * r2; }
    double lin = 0.0;
    for (int a = 0; a < p; ++a) lin += theta[a] * S[a * p + a];
    return lin + 0.5 * sigma * q;
  };
  for (int it = 0; it < iters; ++it) {
    for (int t = 0; t < np; ++t) sv[t] = S[pa[t] * p + pb[t]];
    for (int i = 0; i < np; ++i) { double r2 = 0.0; for (int j = 0; j < np; ++j) r2 += Hw(i, j) * sv[j]; tv[i] = sigma * r2; }
    std::fill(G.begin(), G.end(), 0.0);
    for (int t = 0; t < np; ++t) {
      if (pa[t] == pb[t]) G[pa[t] * p + pa[t]] = tv[t];
      else G[pa[t] * p + pb[t]] = G[pb[t] * p + pa[t]] = 0.5 * tv[t];
    }
    for (int a = 0; a < p; ++a) G[a * p + a] += theta[a];
    std::vector<double> Y((size_t)p * p), m2, Q2;
    for (int i = 0; i < p * p; ++i) Y[i] = S[i] - G[i] / L;
    for (int a = 0; a < p; ++a) for (int b = a + 1; b < p; ++b) { const double av = 0.5 * (Y[a * p + b] + Y[b * p + a]); Y[a * p + b] = Y[b * p + a] = av; }
    jacobi_eigh(Y, p, m2, Q2);
    for (int a = 0; a < p; ++a) for (int b = 0; b < p; ++b) {
      double v = 0.0;
      for (int k = 0; k < p; ++k) v += Q2[a * p + k] * std::max(m2[k], 0.0) * Q2[b * p + k];
      S[a * p + b] = v;
    }
  }
  return gval();
}

// out = 0.5 (zt - za - zb): polarisation  A((v_a v_b^T + v_b v_a^T)/2) from A((v_a+v_b)(v_a+v_b)^T), A(v_a v_a^T), A(v_b v_b^T)
__global__ void k_polar(int64_t m, const double* zt, const double* za, const double* zb, double* out) {
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < m; i += (int64_t)gridDim.x * blockDim.x)
    out[i] = 0.5 * (zt[i] - za[i] - zb[i]);
}
template <typename T> __global__ void k_add2(int64_t N, const T* x, const T* y, T* out) {   // out = x + y
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += (int64_t)gridDim.x * blockDim.x)
    out[i] = (T)((double)x[i] + (double)y[i]);
}

alora_status ensure_ws(alora_ctx* c) {
  if (c->ws) return ALORA_OK;
  c->ws = new (std::nothrow) SolveWorkspace();
  if (!c->ws) return fail(c, ALORA_ENOMEM, "workspace");
  SolveWorkspace* w = c->ws;
  ALORA_CUDA(c, c->pool.alloc((void**)&w->red_part, sizeof(double) * kNStat * kRedBlocks));
  ALORA_CUDA(c, c->pool.alloc((void**)&w->red_out, sizeof(double) * kNStat));
  ALORA_CUDA(c, c->pool.alloc((void**)&w->lb_part, sizeof(double) * kLbW * kRedBlocks));
  ALORA_CUDA(c, c->pool.alloc((void**)&w->lb_out, sizeof(double) * kLbW));
  ALORA_CUDA(c, c->pool.alloc(&w->w, c->esz * c->n));
  ALORA_CUDA(c, c->pool.alloc(&w->ritz, c->esz * c->n));
  ALORA_CUDA(c, c->pool.alloc((void**)&w->lam, sizeof(double) * std::max<int64_t>(1, c->m)));
  ALORA_CUDA(c, c->pool.alloc((void**)&w->z, sizeof(double) * std::max<int64_t>(1, c->m)));
  ALORA_CUDA(c, c->pool.alloc((void**)&w->zv, sizeof(double) * std::max<int64_t>(1, c->m)));
  return ALORA_OK;
}

// up to three dot products in one pass; results on the host (synchronises)
template <typename TX, typename TY>
alora_status dots(alora_ctx* c, int64_t N, int nd, const TX* x0, const TY* y0, const TX* x1, const TY* y1, const TX* x2,
                  const TY* y2, double out[3]) {
  SolveWorkspace* w = c->ws;
  const int grid = (int)std::max<int64_t>(1, std::min<int64_t>((N + kBlock - 1) / kBlock, kRedBlocks));
  k_dots3<TX, TY><<<grid, kBlock, 0, c->stream>>>(N, x0, y0, x1, y1, x2, y2, nd, w->red_part);
  k_reduce_rows<<<1, kBlock, 0, c->stream>>>(w->red_part, grid, w->red_out);
  c->launches += 2;
  ALORA_CUDA(c, cudaMemcpyAsync(c->pinned + 48, w->red_out, sizeof(double) * 3, cudaMemcpyDeviceToHost, c->stream));
  ALORA_CUDA(c, cudaStreamSynchronize(c->stream));
  for (int i = 0; i < nd; ++i) out[i] = c->pinned[48 + i];
  return ALORA_OK;
}
template <typename T> alora_status dot1(alora_ctx* c, int64_t N, const T* x, const T* y, double* out) {
  double o[3];
  alora_status s = dots<T, T>(c, N, 1, x, y, x, y, x, y, o);
  *out = o[0];
  return s;
}

template <typename T>
alora_status lanczos_impl(alora_ctx* c, const double* mu, int kmax, double tol_abs, uint64_t seed, double* theta_out,
                          T* v_out, int* k_used, double* resid_out, int* n_matvec, int p_want = 1,
                          std::vector<double>* thetas = nullptr, T* U_out = nullptr, std::vector<double>* resids = nullptr) {
  alora_status s = ensure_ws(c);
  if (s != ALORA_OK) return s;
  SolveWorkspace* w = c->ws;
  const int64_t n = c->n;
  kmax = (int)std::min<int64_t>(std::max(1, kmax), n);
  if (w->V_cap < kmax) {
    if (w->V) { c->pool.release(w->V); c->pool.release(w->bd_part); c->pool.release(w->cvec); }
    w->bd_chunks = (int)std::max<int64_t>(1, std::min<int64_t>((n + kBlock * 8 - 1) / (kBlock * 8), 256));   // x ceil(k / kBasisJB) blocks
    ALORA_CUDA(c, c->pool.alloc(&w->V, c->esz * (size_t)n * kmax));
    ALORA_CUDA(c, c->pool.alloc((void**)&w->bd_part, sizeof(double) * (size_t)kmax * w->bd_chunks));
    ALORA_CUDA(c, c->pool.alloc((void**)&w->cvec, sizeof(double) * kmax));
    w->V_cap = kmax;
  }
  T* V = (T*)w->V; T* wv = (T*)w->w;
  const int g = ew_grid(c, n);
  k_counter_uniform<T><<<g, 256, 0, c->stream>>>(n, seed, V);
  c->launches++;
  double nrm2;
  s = dot1<T>(c, n, V, V, &nrm2); if (s != ALORA_OK) return s;
  k_scale<T><<<g, 256, 0, c->stream>>>(n, 1.0 / std::sqrt(nrm2), V);
  c->launches++;
  std::vector<double> al, be, sv;
  double theta = 0.0, resid = INFINITY, beta_last = 0.0;
  int k = 0;
  bool conv = false;
  while (true) {
    // one step = 6 launches and ONE synchronisation: matvec (leaves alpha = <v, S v> on the device), three-term
    // recurrence reading alpha there, two classical Gram-Schmidt passes (dots with their reduction fused, combine; the
    // second combine also forms ||w||^2), then alpha and ||w||^2 come back together
    T* vk = V + (int64_t)k * n;
    s = alora_smatvec(c, mu, vk, 1, wv, nullptr); if (s != ALORA_OK) return s;
    if (n_matvec) ++*n_matvec;
    k_axpy2<T><<<2 * g, 256, 0, c->stream>>>(   /* scalar loads, 30 - 32 registers: eight blocks per SM are resident */n, c->mv_dev + ES_GR, vk, k ? be.back() : 0.0, k ? vk - n : (const T*)nullptr, wv);
    c->launches++;
    for (int pass = 0; pass < 2; ++pass) {  // classical Gram-Schmidt against V[0..k], twice
      k_basis_dots<T><<<dim3(w->bd_chunks, (k + 1 + kBasisJB - 1) / kBasisJB), kBlock, 0, c->stream>>>(n, V, wv, w->bd_part, w->bd_chunks, k + 1, w->cvec, c->ticket);
      k_basis_combine<T><<<g, kBlock, 0, c->stream>>>(n, k + 1, V, w->cvec, 1.0, -1.0, wv, w->red_part, pass ? w->red_out : nullptr, c->ticket);
      c->launches += 2;
    }
    ALORA_CUDA(c, cudaMemcpyAsync(c->pinned + 48, w->red_out, sizeof(double), cudaMemcpyDeviceToHost, c->stream));
    ALORA_CUDA(c, cudaMemcpyAsync(c->pinned + 49, c->mv_dev + ES_GR, sizeof(double), cudaMemcpyDeviceToHost, c->stream));
    ALORA_CUDA(c, cudaStreamSynchronize(c->stream));
    const double b2 = c->pinned[48], a = c->pinned[49];
    al.push_back(a);
    const double beta = std::sqrt(b2);
    beta_last = beta;
    ++k;
    tridiag_smallest(al, be, k, theta, sv);
    resid = std::fabs(beta * sv[k - 1]);
    double tnorm = 1e-300;
    for (double x : al) tnorm = std::max(tnorm, std::fabs(x));
    for (double x : be) tnorm = std::max(tnorm, std::fabs(x));
    if (resid <= tol_abs || beta <= 1e-14 * tnorm) { conv = true; break; }
    if (k >= kmax) break;
    be.push_back(beta);
    k_scale_copy<T><<<g, 256, 0, c->stream>>>(n, 1.0 / beta, wv, V + (int64_t)k * n);
    c->launches++;
  }
  if (v_out) {  // Ritz vector V_k s, normalised
    ALORA_CUDA(c, cudaMemcpyAsync(w->cvec, sv.data(), sizeof(double) * k, cudaMemcpyHostToDevice, c->stream));
    k_basis_combine<T><<<g, kBlock, 0, c->stream>>>(n, k, V, w->cvec, 0.0, 1.0, v_out, nullptr, nullptr, nullptr);
    c->launches++;
    double vv;
    s = dot1<T>(c, n, v_out, v_out, &vv); if (s != ALORA_OK) return s;
    k_scale<T><<<g, 256, 0, c->stream>>>(n, 1.0 / std::sqrt(vv), v_out);
    c->launches++;
    ALORA_CUDA(c, cudaStreamSynchronize(c->stream));  // sv is about to go out of scope
  }
  if (p_want > 1 && thetas) {
    // reading 29: the min(p_want, k) smallest Ritz pairs of the same k-step tridiagonal; vector j at U_out + j n
    // (U_out == nullptr: values and residual estimates only)
    if (k > 1 && (int)be.size() >= k) be.resize(k - 1);
    const int pw = std::min(p_want, k);
    thetas->assign(pw, 0.0);
    if (resids) resids->assign(pw, 0.0);
    std::vector<std::vector<double>> found;
    for (int j = 0; j < pw; ++j) {
      std::vector<double> sj;
      tridiag_jth(al, be, k, j, (*thetas)[j], sj, found);
      found.push_back(sj);
      if (resids) (*resids)[j] = std::fabs(beta_last * sj[k - 1]);
      if (!U_out) continue;
      ALORA_CUDA(c, cudaMemcpyAsync(w->cvec, sj.data(), sizeof(double) * k, cudaMemcpyHostToDevice, c->stream));
      T* uj = U_out + (int64_t)j * n;
      k_basis_combine<T><<<g, kBlock, 0, c->stream>>>(n, k, V, w->cvec, 0.0, 1.0, uj, nullptr, nullptr, nullptr);
      c->launches++;
      double vv;
      s = dot1<T>(c, n, uj, uj, &vv); if (s != ALORA_OK) return s;
      k_scale<T><<<g, 256, 0, c->stream>>>(n, 1.0 / std::sqrt(vv), uj);
      c->launches++;
      ALORA_CUDA(c, cudaStreamSynchronize(c->stream));
    }
  }
  ALORA_CUDA(c, cudaGetLastError());
  if (theta_out) *theta_out = theta;
  if (k_used) *k_used = k;
  if (resid_out) *resid_out = resid;
  return conv ? ALORA_OK : ALORA_ENOTCONV;
}

}  // namespace
}  // namespace alora

using namespace alora;

extern "C" void alora_default_params(alora_params* p) {
  if (!p) return;
  p->eps = 1e-5; p->stop_mode = 0; p->T_max = 100; p->tol0 = 1e-2; p->c_in = 0.1; p->tol_min = 1e-7;
  p->it_max = 500; p->lbfgs_mem = 5; p->p_max = 1; p->k_max = 300; p->tau_neg = -1.0; p->tol_eig = -1.0;
  p->gamma = 2.0; p->kappa = 0.25; p->sigma_max = 1e8; p->tau_shrink = 1e-8; p->s_max = 1e6; p->seed = 12345;
  p->stall_tol = 0.0; p->stall_iters = 3; p->pad_ = 0;
}

namespace alora {
__global__ void __launch_bounds__(kBlock) k_dual_terms(int64_t m, const double* y, const double* z, const double* b, double sigma,
                                                       double* lam, double* part) {
  double st[3] = {0.0, 0.0, 0.0};
  for (int64_t i = (int64_t)blockIdx.x * kBlock + threadIdx.x; i < m; i += (int64_t)gridDim.x * kBlock) {
    const double q = z[i] - b[i], yv = y[i], l = yv - sigma * q;
    if (lam) lam[i] = l;
    st[0] += yv * q; st[1] += q * q; st[2] += l * z[i];
  }
  block_reduce_store<3>(st, part + (int64_t)blockIdx.x * kNStat);
}
// sums over the first n_rows rows of row-major X, Y (r columns, leading dimension ld): X.X and X.Y
template <typename T>
__global__ void __launch_bounds__(kBlock) k_rowdots(int64_t n_rows, int r, int64_t ld, const T* X, const T* Y, double* part) {
  double st[3] = {0.0, 0.0, 0.0};
  const int64_t N = n_rows * r;
  for (int64_t i = (int64_t)blockIdx.x * kBlock + threadIdx.x; i < N; i += (int64_t)gridDim.x * kBlock) {
    const int64_t row = i / r, idx = row * ld + (i - row * r);
    const double x = (double)X[idx];
    st[0] += x * x; st[1] += x * (double)Y[idx];
  }
  block_reduce_store<3>(st, part + (int64_t)blockIdx.x * kNStat);
}
}  // namespace alora

namespace {
alora_status fetch_red(alora_ctx* c, int grid, int cnt, double* out) {
  alora::SolveWorkspace* w = c->ws;
  alora::k_reduce_rows<<<1, alora::kBlock, 0, c->stream>>>(w->red_part, grid, w->red_out);
  c->launches++;
  ALORA_CUDA(c, cudaMemcpyAsync(c->pinned + 48, w->red_out, sizeof(double) * 3, cudaMemcpyDeviceToHost, c->stream));
  ALORA_CUDA(c, cudaStreamSynchronize(c->stream));
  for (int i = 0; i < cnt; ++i) out[i] = c->pinned[48 + i];
  return ALORA_OK;
}
}  // namespace

extern "C" alora_status alora_dual_terms(alora_ctx* c, const double* z_dev, double* lam_dev, double out[3]) {
  if (!c || !out || (!z_dev && c->m > 0)) return c ? fail(c, ALORA_EINVAL, "alora_dual_terms: NULL argument") : ALORA_EINVAL;
  if (!c->have_dual) return fail(c, ALORA_ESTATE, "alora_dual_terms before alora_set_dual");
  ALORA_CUDA(c, cudaSetDevice(c->device));
  alora_status s = ensure_ws(c);
  if (s != ALORA_OK) return s;
  out[0] = out[1] = out[2] = 0.0;
  if (c->m == 0) return ALORA_OK;
  const int grid = (int)std::max<int64_t>(1, std::min<int64_t>((c->m + kBlock - 1) / kBlock, kRedBlocks));
  k_dual_terms<<<grid, kBlock, 0, c->stream>>>(c->m, c->y, z_dev, c->b, c->sigma, lam_dev, c->ws->red_part);
  c->launches++;
  return fetch_red(c, grid, 3, out);
}

extern "C" alora_status alora_rowdots(alora_ctx* c, const void* X, const void* Y, int64_t n_rows, int32_t r, int64_t ld, double out[2]) {
  if (!c || !X || !Y || !out || n_rows < 0 || r < 1 || ld < r) return c ? fail(c, ALORA_EINVAL, "alora_rowdots: bad argument") : ALORA_EINVAL;
  ALORA_CUDA(c, cudaSetDevice(c->device));
  alora_status s = ensure_ws(c);
  if (s != ALORA_OK) return s;
  out[0] = out[1] = 0.0;
  if (n_rows == 0) return ALORA_OK;
  const int grid = (int)std::max<int64_t>(1, std::min<int64_t>((n_rows * r + kBlock - 1) / kBlock, kRedBlocks));
  if (c->dtype == ALORA_F32) k_rowdots<float><<<grid, kBlock, 0, c->stream>>>(n_rows, r, ld, (const float*)X, (const float*)Y, c->ws->red_part);
  else k_rowdots<double><<<grid, kBlock, 0, c->stream>>>(n_rows, r, ld, (const double*)X, (const double*)Y, c->ws->red_part);
  c->launches++;
  return fetch_red(c, grid, 2, out);
}

extern "C" void alora_preset_params(alora_params* p, alora_dtype dtype) {
  if (!p) return;
  alora_default_params(p);
  if (dtype == ALORA_F32) { p->it_max = 100; p->stall_tol = 1e-9; p->stall_iters = 3; }
}

extern "C" alora_status alora_lanczos(alora_ctx* c, const double* mu_dev, int32_t kmax, double tol_abs, uint64_t seed,
                                      int32_t p_want, double* theta, void* V_dev, int32_t* p_found, int32_t* k_used,
                                      double* resid) {
  if (!c || kmax < 1 || p_want < 1 || p_want > 8) return c ? fail(c, ALORA_EINVAL, "alora_lanczos: need kmax >= 1 and 1 <= p_want <= 8") : ALORA_EINVAL;
  ALORA_CUDA(c, cudaSetDevice(c->device));
  alora_status s = resolve_mu(c, &mu_dev, "alora_lanczos");
  if (s != ALORA_OK) return s;
  int k = 0;
  double th0 = 0.0, res0 = 0.0;
  std::vector<double> ths, rss;
  if (p_want == 1) {
    s = c->dtype == ALORA_F32
        ? lanczos_impl<float>(c, mu_dev, kmax, tol_abs, seed, &th0, (float*)V_dev, &k, &res0, nullptr)
        : lanczos_impl<double>(c, mu_dev, kmax, tol_abs, seed, &th0, (double*)V_dev, &k, &res0, nullptr);
    ths.assign(1, th0); rss.assign(1, res0);
  } else {
    s = c->dtype == ALORA_F32
        ? lanczos_impl<float>(c, mu_dev, kmax, tol_abs, seed, &th0, (float*)nullptr, &k, &res0, nullptr, p_want, &ths, (float*)V_dev, &rss)
        : lanczos_impl<double>(c, mu_dev, kmax, tol_abs, seed, &th0, (double*)nullptr, &k, &res0, nullptr, p_want, &ths, (double*)V_dev, &rss);
  }
  if (s != ALORA_OK && s != ALORA_ENOTCONV) return s;
  for (size_t j = 0; j < ths.size(); ++j) { if (theta) theta[j] = ths[j]; if (resid) resid[j] = rss[j]; }
  if (p_found) *p_found = (int32_t)ths.size();
  if (k_used) *k_used = k;
  return s;
}

// ---------------------------------------------------------------------------------------------
// alora_solve: Algorithm 1
// ---------------------------------------------------------------------------------------------
namespace alora {
namespace {

// launches k_lbfgs_dots and the copy of its sums into the pinned block (offset kLbPinned); no synchronisation
constexpr int kLbPinned = 64 + 8 * 256;
template <typename T>
alora_status lbfgs_dots_enqueue(alora_ctx* c, int64_t N, int np, bool have_new, double alpha, const T* D, const T* G, const T* Gp,
                                const LbVecs& v, T* Snew, T* Ynew) {
  SolveWorkspace* w = c->ws;
  if (np < 1 || np > kLbMax) return fail(c, ALORA_EINVAL, "lbfgs_dots: too many pairs");
  // A grid-stride kernel is launched with exactly the blocks that are resident at once: a fixed 592 (four per SM) left
  // a partial second wave as soon as three fitted (ncu, config 4: SMs active 79 % of the kernel, 4.1 TB/s).
  int& occ = w->occ_dots[np];
  if (!occ) {
    switch (np) {
#define X(NP) case NP: cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_lbfgs_dots<T, NP>, kBlock, 0); break;
      X(1) X(2) X(3) X(4) X(5) X(6) X(7) X(8)
#undef X
    }
    occ = std::max(1, occ);
  }
  const int grid = (int)std::max<int64_t>(1, std::min<int64_t>((N / (16 / (int64_t)sizeof(T)) + kBlock / 2 - 1) / (kBlock / 2),   // 128 packs per block and pass
                                                               std::min<int64_t>((int64_t)c->num_sms * occ, kRedBlocks)));
  switch (np) {
#define X(NP) case NP: k_lbfgs_dots<T, NP><<<grid, kBlock, 0, c->stream>>>(N, have_new ? 1 : 0, alpha, D, G, Gp, v, Snew, Ynew, w->lb_part, w->lb_out, c->ticket); break;
    X(1) X(2) X(3) X(4) X(5) X(6) X(7) X(8)
#undef X
  }
  c->launches++;
  ALORA_CUDA(c, cudaMemcpyAsync(c->pinned + kLbPinned, w->lb_out, sizeof(double) * kLbW, cudaMemcpyDeviceToHost, c->stream));
  return ALORA_OK;
}
template <typename T>
alora_status lbfgs_combine(alora_ctx* c, int64_t N, int np, const T* G, const LbVecs& v, const LbCoef& cf, T* D) {
  if (np < 1 || np > kLbMax) return fail(c, ALORA_EINVAL, "lbfgs_combine: too many pairs");
  int& occ = c->ws->occ_comb[np];
  if (!occ) {
    switch (np) {
#define X(NP) case NP: cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_lbfgs_combine<T, NP>, kBlock, 0); break;
      X(1) X(2) X(3) X(4) X(5) X(6) X(7) X(8)
#undef X
    }
    occ = std::max(1, occ);
  }
  const int grid = (int)std::max<int64_t>(1, std::min<int64_t>((N / (16 / (int64_t)sizeof(T)) + kBlock - 1) / kBlock, (int64_t)c->num_sms * occ));
  switch (np) {
#define X(NP) case NP: k_lbfgs_combine<T, NP><<<grid, kBlock, 0, c->stream>>>(N, G, v, cf, D); break;
    X(1) X(2) X(3) X(4) X(5) X(6) X(7) X(8)
#undef X
  }
  c->launches++;
  ALORA_CUDA(c, cudaGetLastError());
  return ALORA_OK;
}

template <typename T>
alora_status solve_impl(alora_ctx* c, const alora_params* prm, T* R_user, int32_t* r_inout, int32_t r_cap, double* y,
                        double* sigma_inout, alora_iter_record* log, int32_t log_cap, alora_result* res) {
  const auto t_start = std::chrono::steady_clock::now();
  alora_status s = ensure_ws(c);
  if (s != ALORA_OK) return s;
  SolveWorkspace* w = c->ws;
  const int64_t n = c->n, m = c->m;
  const int A = (int)(16 / sizeof(T));                    // columns are padded (with zeros) to 16-byte rows
  auto pad = [&](int r) { return (r + A - 1) / A * A; };
  const int mem = std::max(0, std::min(prm->lbfgs_mem, kMemMax));
  int r = *r_inout;
  if (r < 1 || r > r_cap) return fail(c, ALORA_EINVAL, "alora_solve: need 1 <= r <= r_cap");
  if (prm->p_max < 1 || prm->p_max > 4) return fail(c, ALORA_EINVAL, "alora_solve: need 1 <= p_max <= 4");
  const int ldcap = pad(r_cap);
  const int64_t elems = n * (int64_t)ldcap;
  const int nslot = mem + 1;                              // one spare slot receives the candidate pair
  const int nbuf = 5 + 2 * nslot;
  static_assert(5 + 2 * (kMemMax + 1) <= SolveWorkspace::kNBuf, "SolveWorkspace::buf too small");
  if (w->buf_elems < elems || w->nbuf < nbuf) {
    for (int i = 0; i < w->nbuf; ++i) { c->pool.release(w->buf[i]); w->buf[i] = nullptr; }
    w->nbuf = 0; w->buf_elems = 0;          // an allocation failure below leaves a consistent (empty) workspace
    for (int i = 0; i < nbuf; ++i) {
      ALORA_CUDA(c, c->pool.alloc(&w->buf[i], sizeof(T) * elems));
      w->nbuf = i + 1;
    }
    w->buf_elems = elems;
  }
  if (!w->gram) {
    ALORA_CUDA(c, c->pool.alloc((void**)&w->gram_part, sizeof(double) * 256 * 256 * 64));
    ALORA_CUDA(c, c->pool.alloc((void**)&w->gram, sizeof(double) * 256 * 256));
    ALORA_CUDA(c, c->pool.alloc((void**)&w->Qdev, sizeof(double) * 256 * 256));
  }
  if (ldcap > 256) return fail(c, ALORA_EINVAL, "alora_solve: r_cap <= 256");
  T* Rw = (T*)w->buf[0]; T* Gw = (T*)w->buf[1]; T* Dw = (T*)w->buf[2]; T* Gp = (T*)w->buf[3]; T* Rtmp = (T*)w->buf[4];
  T** Sb = (T**)&w->buf[5]; T** Yb = (T**)&w->buf[5 + nslot];
  int ld = pad(r);
  int64_t N = n * (int64_t)ld;
  int g = ew_grid(c, N);
  k_repack<T><<<g, 256, 0, c->stream>>>(n, r, R_user, r, Rw, ld);
  c->launches++;

  const double tau_neg = prm->tau_neg >= 0 ? prm->tau_neg : prm->eps;
  const double tol_eig = prm->tol_eig >= 0 ? prm->tol_eig : prm->eps / 10.0;
  const double normC = c->normC, normb = c->normb;
  double sigma = *sigma_inout;
  double infeas_prev = INFINITY, qnorm_prev = INFINITY;
  uint64_t run = 0;
  int n_evals = 0, n_ls = 0, n_mv = 0, outer = 0;
  bool converged = false;
  double kkt[3] = {0, 0, 0};
  double st[8];

  for (int t = 0; t < prm->T_max; ++t) {
    alora_iter_record rec;
    std::memset(&rec, 0, sizeof(rec));
    rec.t = t; rec.sigma = sigma;
    s = alora_set_dual(c, y, sigma); if (s != ALORA_OK) return s;
    // -- 1. inner solve: F <- argmin_F L_rho(FF^T, y)                (Alg. 1 line 4)
    const double tol_t = std::max(prm->tol_min, std::min(prm->tol0, prm->c_in * infeas_prev));
    std::vector<int> pairs;                 // physical slots of the stored pairs, oldest first
    int spare = 0;                          // physical slot that receives the next candidate pair
    std::vector<double> sy(nslot), yy(nslot), alp(nslot);
    std::vector<std::vector<double>> lb_SY(nslot, std::vector<double>(nslot, 0.0)), lb_YY(nslot, std::vector<double>(nslot, 0.0));
    std::vector<double> lb_sg(nslot, 0.0), lb_yg(nslot, 0.0);
    int it = 0, stalled = 0; bool have_prev = false; double alpha = 0.0, gnorm = 0.0;
    while (true) {
      // the evaluation and -- on the fused L-BFGS path -- the dots pass of the iteration are enqueued back to back and
      // their scalars come back with ONE synchronisation (the dots pass needs nothing the host learns from the evaluation)
      const bool fused = mem > 0 && mem < kLbMax;
      std::vector<int> list;
      if (fused) { list = pairs; if (have_prev) list.push_back(spare); }
      const int np = (int)list.size();
      s = alora_eval(c, Rw, ld, ld, Gw, w->z, nullptr); if (s != ALORA_OK) return s;
      s = stats_enqueue(c, ld); if (s != ALORA_OK) return s;
      if (np > 0) {
        LbVecs lv;
        for (int j = 0; j < kLbMax; ++j) { lv.S[j] = Sb[list[j < np ? j : 0]]; lv.Y[j] = Yb[list[j < np ? j : 0]]; }
        s = lbfgs_dots_enqueue<T>(c, N, np, have_prev, alpha, Dw, Gw, Gp, lv, Sb[spare], Yb[spare]); if (s != ALORA_OK) return s;
      }
      ALORA_CUDA(c, cudaStreamSynchronize(c->stream));
      stats_finish(c, ld, st);
      ++rec.n_evals;
      gnorm = std::sqrt(st[4]);
      if (!std::isfinite(st[0]) || !std::isfinite(gnorm)) return fail(c, ALORA_ECUDA, "alora_solve: non-finite f or gradient");
      bool steepest = true;
      if (fused) {
        // ---- L-BFGS in two passes: all dot products of the iteration (and the new pair) in k_lbfgs_dots, the
        //      coefficients of d in span{g, S_j, Y_j} on the host (same recursion as the two-loop form), one combine
        if (np > 0) {
          const double* h = c->pinned + kLbPinned;
          for (int j = 0; j < np; ++j) { lb_sg[list[j]] = h[j]; lb_yg[list[j]] = h[np + j]; }
          if (have_prev) {
            const int slot = spare;
            const double v_sy = h[2 * np + np - 1], v_yy = h[4 * np + np - 1], v_ss = h[5 * np];
            if (v_sy > 1e-10 * std::sqrt(v_ss * v_yy)) {
              for (int j = 0; j < np; ++j) {
                lb_SY[slot][list[j]] = h[2 * np + j];   // S_new . Y_j
                lb_SY[list[j]][slot] = h[3 * np + j];   // S_j . Y_new
                lb_YY[slot][list[j]] = lb_YY[list[j]][slot] = h[4 * np + j];
              }
              sy[slot] = v_sy; yy[slot] = v_yy;
              pairs.push_back(slot);
              if ((int)pairs.size() > mem) { spare = pairs.front(); pairs.erase(pairs.begin()); }
              else { spare = (int)pairs.size(); }
            }
          }
        }
        if (gnorm / (1.0 + normC) <= tol_t || it >= prm->it_max) break;
        if (!pairs.empty()) {
          const int k = (int)pairs.size();
          std::vector<double> al(k), aq(k), bs(k);   // alpha_i; q = g + sum aq_j Y_j; r = gamma q + sum bs_j S_j
          for (int i = k - 1; i >= 0; --i) {
            const int si = pairs[i];
            double sq = lb_sg[si];
            for (int j = i + 1; j < k; ++j) sq += aq[j] * lb_SY[si][pairs[j]];
            al[i] = sq / sy[si];
            aq[i] = -al[i];
          }
          const int nw = pairs.back();
          const double gamma = sy[nw] / yy[nw];
          for (int i = 0; i < k; ++i) {
            const int si = pairs[i];
            double yq = lb_yg[si];
            for (int j = 0; j < k; ++j) yq += aq[j] * lb_YY[si][pairs[j]];
            double yr = gamma * yq;
            for (int j = 0; j < i; ++j) yr += bs[j] * lb_SY[pairs[j]][si];
            bs[i] = al[i] - yr / sy[si];
          }
          LbCoef cf; LbVecs lv;
          cf.cg = -gamma;
          double gd = cf.cg * st[4];
          for (int j = 0; j < kLbMax; ++j) {
            const int sl = pairs[j < k ? j : 0];
            lv.S[j] = Sb[sl]; lv.Y[j] = Yb[sl];
            cf.cs[j] = j < k ? -bs[j] : 0.0;
            cf.cy[j] = j < k ? -gamma * aq[j] : 0.0;
            if (j < k) gd += cf.cs[j] * lb_sg[sl] + cf.cy[j] * lb_yg[sl];
          }
          if (gd < 0.0) {
            s = lbfgs_combine<T>(c, N, k, Gw, lv, cf, Dw); if (s != ALORA_OK) return s;
            steepest = false;
          } else { pairs.clear(); spare = 0; }   // not a descent direction: restart from -G
        }
      } else {
        if (have_prev && mem > 0) {
          const int slot = spare;
          const int gr = (int)std::max<int64_t>(1, std::min<int64_t>((N + kBlock - 1) / kBlock, kRedBlocks));
          k_make_pair<T><<<gr, kBlock, 0, c->stream>>>(N, alpha, Dw, Gw, Gp, Sb[slot], Yb[slot], w->red_part);
          k_reduce_rows<<<1, kBlock, 0, c->stream>>>(w->red_part, gr, w->red_out);
          c->launches += 2;
          ALORA_CUDA(c, cudaMemcpyAsync(c->pinned + 48, w->red_out, sizeof(double) * 3, cudaMemcpyDeviceToHost, c->stream));
          ALORA_CUDA(c, cudaStreamSynchronize(c->stream));
          const double v_sy = c->pinned[48], v_ss = c->pinned[49], v_yy = c->pinned[50];
          if (v_sy > 1e-10 * std::sqrt(v_ss * v_yy)) {
            sy[slot] = v_sy; yy[slot] = v_yy;
            pairs.push_back(slot);
            if ((int)pairs.size() > mem) { spare = pairs.front(); pairs.erase(pairs.begin()); }
            else { spare = (int)pairs.size(); }   // slots 0..mem are handed out in order until the ring is full
          }
        }
        if (gnorm / (1.0 + normC) <= tol_t || it >= prm->it_max) break;
        // direction: two-loop recursion (reading 5); q lives in Dw
        steepest = pairs.empty();
        if (!steepest) {
          ALORA_CUDA(c, cudaMemcpyAsync(Dw, Gw, sizeof(T) * N, cudaMemcpyDeviceToDevice, c->stream));
          for (int i = (int)pairs.size() - 1; i >= 0; --i) {
            const int sl = pairs[i];
            double d; s = dot1<T>(c, N, Sb[sl], Dw, &d); if (s != ALORA_OK) return s;
            alp[sl] = d / sy[sl];
            k_axpy<T><<<g, 256, 0, c->stream>>>(N, -alp[sl], Yb[sl], Dw);
            c->launches++;
          }
          const int nw = pairs.back();
          k_scale<T><<<g, 256, 0, c->stream>>>(N, sy[nw] / yy[nw], Dw);
          c->launches++;
          for (size_t i = 0; i < pairs.size(); ++i) {
            const int sl = pairs[i];
            double d; s = dot1<T>(c, N, Yb[sl], Dw, &d); if (s != ALORA_OK) return s;
            k_axpy<T><<<g, 256, 0, c->stream>>>(N, alp[sl] - d / sy[sl], Sb[sl], Dw);
            c->launches++;
          }
          k_scale<T><<<g, 256, 0, c->stream>>>(N, -1.0, Dw);
          c->launches++;
          double gd; s = dot1<T>(c, N, Gw, Dw, &gd); if (s != ALORA_OK) return s;
          if (gd >= 0.0) { pairs.clear(); spare = 0; steepest = true; }   // not a descent direction: restart from -G
        }
      }
      if (steepest) { k_scale_copy<T><<<g, 256, 0, c->stream>>>(N, -1.0, Gw, Dw); c->launches++; }
      double p[5];
      s = alora_linesearch(c, Rw, Dw, ld, ld, 1, p); if (s != ALORA_OK) return s;   // warm: Rw was just evaluated
      ++n_ls;
      int flag;
      alpha = quartic_argmin(p, &flag);
      if (prm->stall_tol > 0.0) {   // reading 28: the steps no longer decrease f (rounding floor of the evaluation)
        const double dec = -alpha * (p[1] + alpha * (p[2] + alpha * (p[3] + alpha * p[4])));
        stalled = dec <= prm->stall_tol * (1.0 + std::fabs(p[0])) ? stalled + 1 : 0;
        if (stalled >= prm->stall_iters) break;
      }
      std::swap(Gw, Gp);                                   // Gp <- current gradient
      k_axpy<T><<<g, 256, 0, c->stream>>>(N, alpha, Dw, Rw);   // R <- R + alpha D
      c->launches++;
      ++it; have_prev = true;
    }
    rec.inner_iters = it; rec.gnorm = gnorm; rec.f = st[0];
    double cx = st[1], qq = st[3];
    // -- 2./3. lambda = y - sigma q; smallest eigenpair of C - A^*(lambda)   (Alg. 1 line 5)
    k_lambda2<<<ew_grid(c, m), 256, 0, c->stream>>>(m, y, w->z, c->b, sigma, w->lam);
    c->launches++;
    double theta = 0.0, resid = 0.0; int ksteps = 0;
    std::vector<double> thetas;
    if (prm->p_max > 1) {
      if (!w->ritzp) {
        ALORA_CUDA(c, c->pool.alloc(&w->ritzp, c->esz * (size_t)n * 4));
        ALORA_CUDA(c, c->pool.alloc(&w->vtmp, c->esz * (size_t)n));
        ALORA_CUDA(c, c->pool.alloc((void**)&w->cab, sizeof(double) * (size_t)std::max<int64_t>(1, m) * 11));
      }
      s = lanczos_impl<T>(c, w->lam, prm->k_max, tol_eig * (1.0 + normC), prm->seed + run, &theta, (T*)w->ritz, &ksteps, &resid, &n_mv,
                          prm->p_max, &thetas, (T*)w->ritzp);
    } else {
      s = lanczos_impl<T>(c, w->lam, prm->k_max, tol_eig * (1.0 + normC), prm->seed + run, &theta, (T*)w->ritz, &ksteps, &resid, &n_mv);
    }
    ++run;
    if (s != ALORA_OK && s != ALORA_ENOTCONV) return s;
    rec.theta1 = theta; rec.lanczos_steps = ksteps;
    double theta_kkt = theta;
    bool changed = false;
    const bool neg = -theta / (1.0 + normC) > tau_neg;
    if (neg && r + 1 <= r_cap) {
      // -- 4. grow (Alg. 1 lines 6-8), p = 1: s* = -theta / (sigma |A(vv^T)|^2).  At r = r_cap the
      //       step is skipped (reading 27): the dual update and the sigma schedule carry on at rank r_cap.
      // reading 29 (p_max > 1): every Ritz pair of the run that is itself sufficiently negative joins V; S from the
      // small SDP; new columns V S^{1/2}, at most r_cap - r of them (largest eigenvalues of S first)
      int added = 0;
      std::vector<int> sel;
      for (int j = 0; j < (int)thetas.size(); ++j) if (-thetas[j] / (1.0 + normC) > tau_neg) sel.push_back(j);
      if ((int)sel.size() > 1) {
        const int p = (int)sel.size(), np = p * (p + 1) / 2;
        const T* U = (const T*)w->ritzp;
        std::vector<int> pa, pb;
        for (int a = 0; a < p; ++a) for (int b = a; b < p; ++b) { pa.push_back(a); pb.push_back(b); }
        auto cvec = [&](int t) { return w->cab + (size_t)t * std::max<int64_t>(1, m); };
        auto diag_idx = [&](int a) { int t = 0; for (int a2 = 0; a2 < a; ++a2) t += p - a2; return t; };
        for (int a = 0; a < p; ++a) {   // c_aa = A(v_a v_a^T)
          s = alora_eval(c, U + (int64_t)sel[a] * n, 1, 1, nullptr, cvec(diag_idx(a)), nullptr); if (s != ALORA_OK) return s;
        }
        for (int t = 0; t < np; ++t) {
          if (pa[t] == pb[t]) continue;
          k_add2<T><<<ew_grid(c, n), 256, 0, c->stream>>>(n, U + (int64_t)sel[pa[t]] * n, U + (int64_t)sel[pb[t]] * n, (T*)w->vtmp);
          s = alora_eval(c, w->vtmp, 1, 1, nullptr, cvec(10), nullptr); if (s != ALORA_OK) return s;
          k_polar<<<ew_grid(c, m), 256, 0, c->stream>>>(m, cvec(10), cvec(diag_idx(pa[t])), cvec(diag_idx(pb[t])), cvec(t));
          c->launches += 2;
        }
        std::vector<double> H((size_t)np * np, 0.0);
        for (int i = 0; i < np; ++i)
          for (int j = i; j < np; ++j) {
            double d3[3];
            s = dots<double, double>(c, m, 1, cvec(i), cvec(j), cvec(i), cvec(j), cvec(i), cvec(j), d3); if (s != ALORA_OK) return s;
            H[(size_t)i * np + j] = H[(size_t)j * np + i] = d3[0];
          }
        std::vector<double> th(p), S;
        for (int a = 0; a < p; ++a) th[a] = thetas[sel[a]];
        const double gv = growth_sdp_host(p, th.data(), H, sigma, S);
        if (gv < 0.0) {
          std::vector<double> mu, Q;
          std::vector<double> S2(S);
          jacobi_eigh(S2, p, mu, Q);
          std::vector<int> cols;
          for (int k2 = p - 1; k2 >= 0; --k2) if (mu[k2] > 1e-12 * mu[p - 1] && (int)cols.size() < r_cap - r) cols.push_back(k2);
          const int ld2 = pad(r + (int)cols.size());
          if (ld2 != ld) {
            k_repack<T><<<ew_grid(c, n * (int64_t)ld2), 256, 0, c->stream>>>(n, r, Rw, ld, Rtmp, ld2);
            c->launches++;
            std::swap(Rw, Rtmp);
            ld = ld2;
          }
          for (int k2 : cols) {   // column = sum_a v_a Q[a][k2] sqrt(mu_k2)
            ALORA_CUDA(c, cudaStreamSynchronize(c->stream));
            k_scale_copy<T><<<ew_grid(c, n), 256, 0, c->stream>>>(n, Q[0 * p + k2] * std::sqrt(mu[k2]), U + (int64_t)sel[0] * n, (T*)w->vtmp);
            for (int a = 1; a < p; ++a)
              k_axpy<T><<<ew_grid(c, n), 256, 0, c->stream>>>(n, Q[a * p + k2] * std::sqrt(mu[k2]), U + (int64_t)sel[a] * n, (T*)w->vtmp);
            k_set_col<T><<<ew_grid(c, n), 256, 0, c->stream>>>(n, ld, r + added, 1.0, (const T*)w->vtmp, Rw);
            c->launches += p + 1;
            ++added;
          }
        }
      }
      if (added == 0) {   // p = 1 closed form
        s = alora_eval(c, w->ritz, 1, 1, nullptr, w->zv, nullptr); if (s != ALORA_OK) return s;
        double avv[3]; s = dots<double, double>(c, m, 1, w->zv, w->zv, w->zv, w->zv, w->zv, w->zv, avv); if (s != ALORA_OK) return s;
        const double den = sigma * avv[0];
        const double s_star = (den > 0.0 && -theta / den < prm->s_max) ? -theta / den : prm->s_max;
        const int ld2 = pad(r + 1);
        if (ld2 != ld) {
          k_repack<T><<<ew_grid(c, n * (int64_t)ld2), 256, 0, c->stream>>>(n, r, Rw, ld, Rtmp, ld2);
          c->launches++;
          std::swap(Rw, Rtmp);
          ld = ld2;
        }
        k_set_col<T><<<ew_grid(c, n), 256, 0, c->stream>>>(n, ld, r, std::sqrt(s_star), (const T*)w->ritz, Rw);
        c->launches++;
        added = 1;
      }
      r += added; rec.grew = added; changed = true;
    } else if (!neg && r > 1) {
      // -- 5. shrink (reading 13): drop the numerically null directions of R
      const int nblk = (int)std::max<int64_t>(1, std::min<int64_t>(64, n / 256));
      const int64_t rpb = (n + nblk - 1) / nblk;
      k_gram<T><<<nblk, 256, 0, c->stream>>>(n, r, Rw, ld, w->gram_part, rpb);
      k_gram_reduce<<<(r * r + 255) / 256, 256, 0, c->stream>>>(w->gram_part, nblk, r * r, w->gram);
      c->launches += 2;
      std::vector<double> M((size_t)r * r), mu, Q;
      ALORA_CUDA(c, cudaMemcpyAsync(M.data(), w->gram, sizeof(double) * r * r, cudaMemcpyDeviceToHost, c->stream));
      ALORA_CUDA(c, cudaStreamSynchronize(c->stream));
      jacobi_eigh(M, r, mu, Q);
      int first_keep = 0;
      while (first_keep < r && !(mu[first_keep] > prm->tau_shrink * mu[r - 1])) ++first_keep;
      const int rk = r - first_keep;
      if (first_keep > 0 && rk >= 1) {
        std::vector<double> Qk((size_t)r * rk);
        for (int i = 0; i < r; ++i) for (int cidx = 0; cidx < rk; ++cidx) Qk[(size_t)i * rk + cidx] = Q[(size_t)i * r + first_keep + cidx];
        ALORA_CUDA(c, cudaMemcpyAsync(w->Qdev, Qk.data(), sizeof(double) * r * rk, cudaMemcpyHostToDevice, c->stream));
        const int ld2 = pad(rk);
        k_rotate<T><<<ew_grid(c, n * (int64_t)ld2), 256, 0, c->stream>>>(n, r, rk, Rw, ld, w->Qdev, Rtmp, ld2);
        c->launches++;
        ALORA_CUDA(c, cudaStreamSynchronize(c->stream));
        std::swap(Rw, Rtmp);
        rec.shrank = first_keep; r = rk; ld = ld2; changed = true;
      }
    }
    if (changed) {
      N = n * (int64_t)ld; g = ew_grid(c, N);
      s = alora_eval(c, Rw, ld, ld, nullptr, w->z, st); if (s != ALORA_OK) return s;   // q, <C,X> at the new R
      cx = st[1]; qq = st[3];
    }
    const double qnorm = std::sqrt(qq);
    // -- 6. y <- y + rho (b - A FF^T)                               (Alg. 1 line 10)
    k_dual_update<<<ew_grid(c, m), 256, 0, c->stream>>>(m, sigma, w->z, c->b, y);
    c->launches++;
    if (changed) {  // reading 17: S(lambda) != S(y_new) once R changed
      int k2 = 0;
      s = lanczos_impl<T>(c, y, prm->k_max, tol_eig * (1.0 + normC), prm->seed + run, &theta_kkt, (T*)nullptr, &k2, &resid, &n_mv);
      ++run;
      if (s != ALORA_OK && s != ALORA_ENOTCONV) return s;
    }
    double by[3]; s = dots<double, double>(c, m, 1, c->b, y, c->b, y, c->b, y, by); if (s != ALORA_OK) return s;
    kkt[0] = qnorm / (1.0 + normb);
    kkt[1] = std::fabs(std::min(0.0, theta_kkt)) / (1.0 + normC);
    kkt[2] = std::fabs(cx - by[0]) / (1.0 + std::fabs(cx) + std::fabs(by[0]));
    rec.r = r; rec.cx = cx; rec.qnorm = qnorm; rec.kkt[0] = kkt[0]; rec.kkt[1] = kkt[1]; rec.kkt[2] = kkt[2];
    // -- 7. sigma schedule (reading 12)
    if (qnorm > prm->kappa * qnorm_prev && kkt[0] > prm->eps) sigma = std::min(prm->gamma * sigma, prm->sigma_max);
    qnorm_prev = qnorm; infeas_prev = kkt[0];
    if (log && t < log_cap) log[t] = rec;
    n_evals += rec.n_evals; outer = t + 1;
    // -- 8. until KKT(FF^T, y) <= eps                                (Alg. 1 line 11, eq. 77)
    const bool done = prm->stop_mode == 1 ? kkt[0] <= prm->eps : std::max(kkt[0], std::max(kkt[1], kkt[2])) <= prm->eps;
    if (done) { converged = true; break; }
  }
  // hand the state back: R (n x r, ld = r), r, y (updated in place), sigma
  k_repack<T><<<ew_grid(c, n * (int64_t)r), 256, 0, c->stream>>>(n, r, Rw, ld, R_user, r);
  c->launches++;
  ALORA_CUDA(c, cudaStreamSynchronize(c->stream));
  ALORA_CUDA(c, cudaGetLastError());
  *r_inout = r; *sigma_inout = sigma;
  if (res) {
    res->converged = converged; res->outer_iters = outer; res->n_evals = n_evals; res->n_linesearch = n_ls;
    res->n_matvec = n_mv; res->r_final = r; res->kkt[0] = kkt[0]; res->kkt[1] = kkt[1]; res->kkt[2] = kkt[2];
    res->sigma_final = sigma;
    res->seconds = std::chrono::duration<double>(std::chrono::steady_clock::now() - t_start).count();
  }
  return converged ? ALORA_OK : ALORA_ENOTCONV;
}

}  // namespace
}  // namespace alora

extern "C" alora_status alora_solve(alora_ctx* c, const alora_params* prm, void* R_dev, int32_t* r_inout, int32_t r_cap,
                                    double* y_dev, double* sigma_inout, alora_iter_record* log, int32_t log_cap,
                                    alora_result* res) {
  if (!c || !prm || !R_dev || !r_inout || !sigma_inout || (!y_dev && c->m > 0))
    return c ? fail(c, ALORA_EINVAL, "alora_solve: NULL argument") : ALORA_EINVAL;
  if (!(*sigma_inout > 0.0)) return fail(c, ALORA_EINVAL, "alora_solve: sigma > 0");
  ALORA_CUDA(c, cudaSetDevice(c->device));
  return c->dtype == ALORA_F32
      ? solve_impl<float>(c, prm, (float*)R_dev, r_inout, r_cap, y_dev, sigma_inout, log, log_cap, res)
      : solve_impl<double>(c, prm, (double*)R_dev, r_inout, r_cap, y_dev, sigma_inout, log, log_cap, res);
}
